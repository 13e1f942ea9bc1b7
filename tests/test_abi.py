"""The C-ABI library loads and exports every symbol include/cdz.h declares (no compute, CPU only)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2604_19718_b200 import build

    return build.build()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "cdz.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cdz_[a-z0-9_]+)\s*\(", src)))


def test_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    names = declared_symbols()
    assert len(names) >= 20
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/cdz.h but not exported"
    from paper_2604_19718_b200 import binding

    assert sorted(binding.EXPORTS) == names


def test_host_only_calls(libpath):
    """TT builder and argument validation run on the host; no CUDA device is touched."""
    from paper_2604_19718_b200 import binding as B
    from paper_2604_19718_b200 import inputs as I

    tt = B.TensorTrain.build("PPTWVRLATTIWWMTFILCS", B.TT_SINGLE_CODON, I.codon_logw(1000))
    sigma, counts, nops = tt.describe()
    assert tt.n == 60 and sum(sigma[:-1]) == 106 and sigma[0] == 1 and sigma[-1] == 1
    tt2 = B.TensorTrain.build("WGVSQPIRWI", B.TT_CODON_PAIR, I.codon_logw(5000), I.pair_logw(5000))
    s2, c2, _ = tt2.describe()
    assert sum(s2[:-1]) == 100 and s2[-1] == 3
    with pytest.raises(B.CdzError):
        B.TensorTrain.build("PPXW", B.TT_SINGLE_CODON)
    with pytest.raises(B.CdzError):
        bad = I.codon_logw(1).copy()
        bad[3] = float("nan")
        B.TensorTrain.build("PPW", B.TT_SINGLE_CODON, bad)
    m = I.nn_model()
    B.Model(m)
    m.max_interior = 31
    with pytest.raises(B.CdzError):
        B.Model(m)
    assert tt.workspace_bytes() > 0


def test_tt_matches_oracle_operator_lists(libpath):
    """Both sides build the same operator lists (PAPER.md S3c) independently."""
    import ctypes as C

    from oracle import oracle as O
    from paper_2604_19718_b200 import binding as B
    from paper_2604_19718_b200 import inputs as I

    for cfg, L in ((1, 20), (2, 25), (5, 30)):
        d = I.design(cfg, 0, L)
        sig_o, ops_o = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw).get()
        tt = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
        sig, counts, nops = tt.describe()
        assert sig == sig_o and counts == [len(o) for o in ops_o]
