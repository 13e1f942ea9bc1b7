"""SURVEY 8f-2 (eq 2.8, S4d lines 245-260, Alg S4.5): minimisation over sequences and structures in
the tropical (min, +) semiring through the C ABI (`cdz_mfe`), against the oracle's tropical recursion (`orc_mfe`, itself pinned to
explicit enumeration of every operator path and structure) and against properties that hold at any size: the returned state is a
coding sequence with a valid structure whose own free energy (evaluated by the oracle's energy function) IS f_min, f_min >= -log Z,
and no sampled state lies below it.  Several minimisers may exist: the value is compared, the state is validated."""
import numpy as np
import pytest

from paper_2604_19718_b200 import inputs as I

pytestmark = pytest.mark.gpu
RTOL = 1e-9


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding, build

    build.build()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle

    return oracle


def _check(B, O, m, tt_g, tt_o, want=None):
    f, seq, pair = B.mfe(B.Model(m), tt_g)
    seq, pair = seq.cpu().numpy(), pair.cpu().numpy()
    if want is not None:
        assert abs(f - want) <= RTOL * max(1.0, abs(want)), (f, want)
    assert (seq < 4).all()
    lw = O.logweight(m, tt_o, seq, pair)  # -inf if the state is not in the ensemble
    assert np.isfinite(lw) and abs(-lw - f) <= RTOL * max(1.0, abs(f)), (f, lw)
    return f, seq, pair


@pytest.mark.parametrize("aa,kind,cw,pw", [("MW", 0, 0, 0), ("LSR", 0, 1, 0), ("LSR", 1, 1, 1), ("RSLG", 0, 1, 0), ("GRL", 1, 1, 1),
                                            ("MWFMWM", 0, 1, 0)])
def test_mfe_equals_enumeration_and_oracle(B, O, aa, kind, cw, pw):
    m = I.tm1_model()
    m.ml_a = 0.4
    cwv, pwv = (I.tm1_codon_logw() if cw else None), (I.tm1_pair_logw() if pw else None)
    tto = O.TT.build(aa, kind, cwv, pwv)
    fb, _, _ = O.mfe(m, tto, brute=True)
    fo, _, _ = O.mfe(m, tto)
    assert abs(fo - fb) < 1e-12 * max(1.0, abs(fb))
    _check(B, O, m, B.TensorTrain.build(aa, kind, cwv, pwv), tto, want=fb)


@pytest.mark.parametrize("cfg,L", [(1, 13), (1, 20), (2, 12), (5, 14), (1, 40), (5, 30)])
def test_mfe_equals_oracle_baseline_designs(B, O, cfg, L):
    """Prefixes of the BASELINE designs and the whole config 1 (NN model; all loop types, multiloops, both tensor trains)."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    tto = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    fo, so, po = O.mfe(m, tto)
    f, seq, pair = _check(B, O, m, B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw), tto, want=fo)
    assert f >= -O.inside(m, tto).logZ - 1e-9


def test_mfe_generic_operators_bond_dimension_8(B, O):
    m = I.tm1_model()
    m.allow_all_pairs = 1
    ops = I.closed_form_inputs("zero8", 18)
    tto = O.TT.from_ops(ops)
    fo, _, _ = O.mfe(m, tto)
    _check(B, O, m, B.TensorTrain.from_operators(ops), tto, want=fo)


@pytest.mark.parametrize("cfg,L", [(5, 150), (2, 300), (4, 1000)])
def test_mfe_properties_at_size(B, O, cfg, L):
    """450 / 900 / 3000 nt: the minimiser is a valid state that attains f_min; f_min >= -log Z of the same design; none of 64 exact
    samples lies below it; the run is deterministic."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    ttg = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    tto = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    f, seq, pair = _check(B, O, m, ttg, tto)
    tab, lz = B.inside(B.Model(m), ttg)
    assert f >= -lz - 1e-9 * abs(lz)
    s, p = tab.sample(64, d.sample_seed)
    s, p = s.cpu().numpy(), p.cpu().numpy()
    for k in range(0, 64, 4):
        assert -O.logweight(m, tto, s[k], p[k]) >= f - 1e-9 * abs(f)
    f2, _, _ = B.mfe(B.Model(m), ttg, traceback=False)
    assert f2 == f
    print(f"config {cfg} L={L}: f_min = {f:.6f} kT, -log Z = {-lz:.6f}, pairs in the minimiser: {(pair >= 0).sum() // 2}")
