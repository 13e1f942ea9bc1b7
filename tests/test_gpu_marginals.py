"""GPU parity of the outside pass (base-pair probabilities, eq 2.5 line 85 / eq 4.1) through
the C ABI (`cdz_marginals`): element-wise against the oracle's definition-level marginals (`orc_marginals`: ratios of restricted
partition functions, itself pinned to brute force) at sizes the oracle finishes, and against sum rules and the frequencies of
the (bit-exact) sampler at the BASELINE sizes."""
import math

import numpy as np
import pytest

from paper_2604_19718_b200 import inputs as I

pytestmark = pytest.mark.gpu
BPP_ATOL = 1e-10  # probabilities; fp64 sums of <= 1e5 positive terms, log Z agrees to 1e-12 relative


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding, build

    build.build()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle

    return oracle


def _gpu_bpp(B, m, aa, kind, cw, pw):
    tg, lz = B.inside(B.Model(m), B.TensorTrain.build(aa, kind, cw, pw))
    return tg, lz, tg.marginals().cpu().numpy()


@pytest.mark.parametrize("aa,kind", [("RSLG", 0), ("LSR", 1), ("MFL", 1), ("GRL", 0), ("MW", 0), ("LLLLL", 1), ("MRSLGWLS", 0)])
def test_bpp_equals_oracle_tm1(B, O, aa, kind):
    """Every entry of the pair matrix and the unpaired diagonal against the oracle (mismatch-rich test model, all loop types)."""
    m = I.tm1_model()
    m.ml_a = 0.4
    cw, pw = I.tm1_codon_logw(), (I.tm1_pair_logw() if kind else None)
    bo, _, _ = O.inside(m, O.TT.build(aa, kind, cw, pw)).marginals()
    _, _, bg = _gpu_bpp(B, m, aa, kind, cw, pw)
    np.testing.assert_allclose(bg, bo, atol=BPP_ATOL, rtol=0)
    assert (np.tril(bg, -1) == 0).all()


@pytest.mark.parametrize("cfg,L", [(1, 8), (1, 13), (2, 9), (5, 10)])
def test_bpp_equals_oracle_baseline_prefixes(B, O, cfg, L):
    """Prefixes of the BASELINE designs (NN model of configs[0]; single-codon and codon-pair TT): n = 24 .. 39."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    bo, _, _ = O.inside(m, O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)).marginals()
    _, _, bg = _gpu_bpp(B, m, d.aa, d.kind, d.codon_logw, d.pair_logw)
    np.testing.assert_allclose(bg, bo, atol=BPP_ATOL, rtol=0)


def test_bpp_generic_operators_bond_dimension_8(B, O):
    """cdz_tt_from_operators at the kernel limits (bond dimension 8, 16 boundary states), all pairs allowed."""
    m = I.tm1_model()
    n = 16
    ops = []
    for i in range(n):
        sa = 1 if i == 0 else 8
        sc = 1 if i == n - 1 else 8
        pos = []
        for a in range(sa):
            for b in (i % 4, (i + 1) % 4):
                c = (a + 3 * b + i) % sc
                pos.append((a, b, c, 0.5 + 0.03 * ((3 * a + 5 * b + i) % 11)))
        ops.append(pos)
    bo, _, _ = O.inside(m, O.TT.from_ops(ops)).marginals()
    tg, _ = B.inside(B.Model(m), B.TensorTrain.from_operators(ops))
    np.testing.assert_allclose(tg.marginals().cpu().numpy(), bo, atol=BPP_ATOL, rtol=0)


@pytest.mark.parametrize("cfg,L,J", [(1, 20, 40000), (5, 150, 4000), (2, 300, 2000)])
def test_bpp_sum_rules_and_sample_frequencies(B, cfg, L, J):
    """Whole config 1 (60 nt), config 5 item 0 (450 nt) and config 2 (900 nt, both codon-pair TT): 0 <= P <= 1, rows + unpaired = 1 by construction, every
    P(i.j) within 6 sigma of its frequency among J exact samples, and the expected number of pairs matches the sample mean."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    tg, lz, bg = _gpu_bpp(B, m, d.aa, d.kind, d.codon_logw, d.pair_logw)
    n = 3 * L
    P = np.triu(bg, 1)
    assert (P >= 0).all() and (P <= 1 + 1e-12).all()
    un = np.diag(bg)
    assert (un >= -1e-9).all() and (un <= 1 + 1e-12).all()
    np.testing.assert_allclose((P + P.T).sum(1) + un, 1.0, atol=1e-12)
    _, pair = tg.sample(J, d.sample_seed)
    pair = pair.cpu().numpy()
    freq = np.zeros((n, n))
    for i in range(n):
        col = pair[:, i]
        sel = col > i
        np.add.at(freq[i], col[sel], 1.0)
    freq /= J
    sig = np.sqrt(np.maximum(P * (1 - P), 1.0 / J) / J)
    assert (np.abs(freq - P) <= 6 * sig + 1e-12).all()
    npairs = (pair > np.arange(n)[None, :]).sum(1)
    assert abs(npairs.mean() - P.sum()) <= 6 * npairs.std() / math.sqrt(J) + 1e-9
    np.testing.assert_allclose((pair < 0).mean(0), un, atol=6 * 0.5 / math.sqrt(J))


def test_marginals_call_contract(B):
    """Before the inside pass the call is a state error; base / codon buffers are rejected (not built)."""
    import ctypes as C

    import torch

    tt = B.TensorTrain.build("M", 0)
    tab, _ = B.inside(B.Model(I.nn_model()), tt)
    buf = torch.zeros(3 * 3, dtype=torch.float64, device="cuda")
    base = torch.zeros(3 * 4, dtype=torch.float64, device="cuda")
    L = B.lib()
    assert L.cdz_marginals(tab.h, C.c_void_p(buf.data_ptr()), C.c_void_p(base.data_ptr()), None, None) < 0
    assert (buf == 0).all()
    assert L.cdz_marginals(tab.h, C.c_void_p(buf.data_ptr()), None, None, None) == 0
    torch.cuda.synchronize()
    b = buf.cpu().numpy().reshape(3, 3)
    np.testing.assert_allclose(b, np.eye(3), atol=1e-12)  # n = 3: nothing can pair
