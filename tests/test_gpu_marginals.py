"""GPU parity of the outside pass through the C ABI (`cdz_marginals`): base-pair probabilities (eq 2.5 line 85 /
eq 4.1), base marginals (eq 2.6 line 90 / eq 4.2) and codon marginals (eq 2.7 line 96 / eq 4.3), element-wise
against the oracle's definition-level marginals (`orc_marginals`: ratios of restricted partition functions, itself pinned to brute
force) at sizes the oracle finishes, against stored oracle values at config 1, and against sum rules and the frequencies of the
(bit-exact) sampler at the BASELINE sizes."""
import math
import os

import numpy as np
import pytest

from paper_2604_19718_b200 import inputs as I

pytestmark = pytest.mark.gpu
ATOL = 1e-10  # probabilities; fp64 sums of <= 1e5 positive terms, log Z agrees to 1e-12 relative
GOLD = os.path.join(os.path.dirname(__file__), "golden")
CODE = "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF"


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding, build

    build.build()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle

    return oracle


def _gpu(B, m, aa, kind, cw, pw, **kw):
    tg, lz = B.inside(B.Model(m), B.TensorTrain.build(aa, kind, cw, pw))
    bpp, base, codon = tg.marginals(**kw)
    return tg, lz, bpp.cpu().numpy(), base.cpu().numpy(), codon.cpu().numpy()


def _check_rules(aa, bpp, base, codon):
    """What holds at any size: probabilities in [0,1]; the pair matrix with the (independently computed) unpaired diagonal is doubly
    stochastic; base and codon marginals are normalised; foreign codons carry exactly zero mass; the base
    marginals are the codon marginals summed per nucleotide."""
    n = bpp.shape[0]
    P = np.triu(bpp, 1)
    assert (np.tril(bpp, -1) == 0).all()
    assert (P >= -1e-12).all() and (P <= 1 + 1e-12).all()
    np.testing.assert_allclose((P + P.T).sum(1) + np.diag(bpp), 1.0, atol=1e-9)
    np.testing.assert_allclose(base.sum(1), 1.0, atol=1e-9)
    np.testing.assert_allclose(codon.sum(1), 1.0, atol=1e-9)
    assert (base >= -1e-12).all() and (codon >= -1e-12).all()
    for k, a in enumerate(aa):
        foreign = np.array([CODE[c] != a for c in range(64)])
        assert (codon[k][foreign] == 0.0).all()
    sel = np.zeros((3, 4, 64))
    for c in range(64):
        for pos in range(3):
            sel[pos, (c >> (2 * (2 - pos))) & 3, c] = 1.0
    from_codon = np.einsum("pbc,kc->kpb", sel, codon).reshape(n, 4)
    np.testing.assert_allclose(from_codon, base, atol=1e-9)


@pytest.mark.parametrize("aa,kind", [("RSLG", 0), ("LSR", 1), ("MFL", 1), ("GRL", 0), ("MW", 0), ("LLLLL", 1), ("MRSLGWLS", 0)])
def test_marginals_equal_oracle_tm1(B, O, aa, kind):
    """Every entry of the pair matrix, the unpaired diagonal, the base and the codon marginals against the oracle (mismatch-rich test
    model, all loop types)."""
    m = I.tm1_model()
    m.ml_a = 0.4
    cw, pw = I.tm1_codon_logw(), (I.tm1_pair_logw() if kind else None)
    bo, so, co = O.inside(m, O.TT.build(aa, kind, cw, pw)).marginals()
    _, _, bg, sg, cg = _gpu(B, m, aa, kind, cw, pw)
    np.testing.assert_allclose(bg, bo, atol=ATOL, rtol=0)
    np.testing.assert_allclose(sg, so, atol=ATOL, rtol=0)
    np.testing.assert_allclose(cg, co, atol=ATOL, rtol=0)
    _check_rules(aa, bg, sg, cg)


@pytest.mark.parametrize("cfg,L", [(1, 8), (1, 12), (2, 9), (5, 8)])
def test_marginals_equal_oracle_baseline_prefixes(B, O, cfg, L):
    """Prefixes of the BASELINE designs (NN model of configs[0]; single-codon and codon-pair TT): n = 24 .. 36 (the oracle takes O(n^2)
    restricted inside passes: minutes at 36 nt)."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    bo, so, co = O.inside(m, O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)).marginals()
    _, _, bg, sg, cg = _gpu(B, m, d.aa, d.kind, d.codon_logw, d.pair_logw)
    np.testing.assert_allclose(bg, bo, atol=ATOL, rtol=0)
    np.testing.assert_allclose(sg, so, atol=ATOL, rtol=0)
    np.testing.assert_allclose(cg, co, atol=ATOL, rtol=0)
    _check_rules(d.aa, bg, sg, cg)


def test_marginals_per_position_codon_weights(B, O):
    """cdz_tt_build_pos: per-residue codon tables, log Z and marginals against the oracle."""
    m = I.tm1_model()
    aa = "RSLGSM"
    rng = np.random.default_rng(11)
    cwp = rng.normal(0.0, 0.5, (len(aa), 64))
    for kind, pw in ((0, None), (1, I.tm1_pair_logw())):
        to = O.inside(m, O.TT.build(aa, kind, cwp, pw))
        bo, so, co = to.marginals()
        tg, lz, bg, sg, cg = _gpu(B, m, aa, kind, cwp, pw)
        assert abs(lz - to.logZ) <= 1e-9 * abs(to.logZ)
        np.testing.assert_allclose(bg, bo, atol=ATOL, rtol=0)
        np.testing.assert_allclose(cg, co, atol=ATOL, rtol=0)
        np.testing.assert_allclose(sg, so, atol=ATOL, rtol=0)


def test_marginals_generic_operators_bond_dimension_8(B, O):
    """cdz_tt_from_operators at the kernel limits (bond dimension 8, 16 boundary states), all pairs allowed: pair matrix and base
    marginals (a generic operator list has no codon labels: codon_dev is rejected)."""
    m = I.tm1_model()
    m.allow_all_pairs = 1
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
    bo, so, _ = O.inside(m, O.TT.from_ops(ops)).marginals()
    tg, _ = B.inside(B.Model(m), B.TensorTrain.from_operators(ops))
    bg, sg, _ = tg.marginals(codon=False)
    np.testing.assert_allclose(bg.cpu().numpy(), bo, atol=ATOL, rtol=0)
    np.testing.assert_allclose(sg.cpu().numpy(), so, atol=ATOL, rtol=0)
    with pytest.raises(B.CdzError):
        tg.marginals()


def _stored_marginals(cfg):
    path = os.path.join(GOLD, f"oracle_marginals_config{cfg}.txt")
    if not os.path.exists(path):
        return None
    d = I.design(cfg, 0)
    n = d.n
    bpp, base, codon = np.zeros((n, n)), np.zeros((n, 4)), np.zeros((n // 3, 64))
    for ln in open(path):
        if ln.startswith("#") or not ln.strip():
            continue
        kind, a, b, v = ln.split()
        {"bpp": bpp, "base": base, "codon": codon}[kind][int(a), int(b)] = float(v)
    return bpp, base, codon


def test_config1_full_marginals_vs_stored_oracle(B):
    """Whole config 1 (60 nt): every P(i.j), unpaired probability, base and codon marginal against the values orc_marginals computed for
    this design (tests/golden/oracle_marginals_config1.txt, written by tests/golden/make_golden.py marginals 1; oracle only)."""
    gold = _stored_marginals(1)
    if gold is None:
        pytest.skip("tests/golden/oracle_marginals_config1.txt not generated")
    d = I.design(1, 0)
    _, _, bg, sg, cg = _gpu(B, I.nn_model(), d.aa, d.kind, d.codon_logw, d.pair_logw)
    np.testing.assert_allclose(bg, gold[0], atol=ATOL, rtol=0)
    np.testing.assert_allclose(sg, gold[1], atol=ATOL, rtol=0)
    np.testing.assert_allclose(cg, gold[2], atol=ATOL, rtol=0)


def _chi2_pvalue(stat, dof):
    """Wilson-Hilferty normal approximation of the chi-square survival function (no scipy dependence in the GPU tests)."""
    if dof <= 0:
        return 1.0
    z = ((stat / dof) ** (1.0 / 3.0) - (1.0 - 2.0 / (9.0 * dof))) / math.sqrt(2.0 / (9.0 * dof))
    return 0.5 * math.erfc(z / math.sqrt(2.0))


@pytest.mark.parametrize("cfg,L,J", [(1, 20, 40000), (5, 150, 4000), (2, 300, 2000)])
def test_sum_rules_and_sample_frequencies(B, cfg, L, J):
    """Whole config 1 (60 nt), config 5 item 0 (450 nt) and config 2 (900 nt, both codon-pair TT): the rules of _check_rules (none of
    them holds by construction: the unpaired diagonal and the base / codon marginals come from the operator usages); every P(i.j)
    within 6 sigma of its frequency among J exact samples; chi-square of the sampled codon frequencies against the exact codon
    marginals (SURVEY c-16: categories with expected count < 5 pooled per position, global statistic, p > 1e-3); unpaired
    frequency of every position against the exact unpaired probability."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    tg, lz, bg, sg, cg = _gpu(B, m, d.aa, d.kind, d.codon_logw, d.pair_logw)
    n = 3 * L
    _check_rules(d.aa, bg, sg, cg)
    P = np.triu(bg, 1)
    un = np.diag(bg)
    seq, pair = tg.sample(J, d.sample_seed)
    seq, pair = seq.cpu().numpy(), pair.cpu().numpy()
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
    # codon chi-square against the exact marginals
    stat, dof = 0.0, 0
    for k in range(L):
        cod = 16 * seq[:, 3 * k].astype(int) + 4 * seq[:, 3 * k + 1] + seq[:, 3 * k + 2]
        obs = np.bincount(cod, minlength=64).astype(float)
        assert obs[cg[k] == 0].sum() == 0  # zero mass on disallowed codons
        e = J * cg[k]
        big = e >= 5
        small_e, small_o = e[~big].sum(), obs[~big].sum()
        cats_e, cats_o = list(e[big]), list(obs[big])
        if small_e >= 5:
            cats_e.append(small_e)
            cats_o.append(small_o)
        if len(cats_e) >= 2:
            ce, co = np.array(cats_e), np.array(cats_o)
            stat += ((co - ce) ** 2 / ce).sum()
            dof += len(ce) - 1
    assert _chi2_pvalue(stat, dof) > 1e-3, (stat, dof)
    # paired / unpaired per position.  Pairedness is strongly correlated along a stem, so the per-position statistics are not
    # independent and their sum is not chi-square distributed; each position is tested on its own (5 sigma, n positions).
    fu = (pair < 0).mean(0)
    sig_u = np.sqrt(np.maximum(un * (1 - un), 1.0 / J) / J)
    assert (np.abs(fu - un) <= 5 * sig_u + 1e-12).all()


def test_marginals_library_workspace_and_other_stream(B):
    """workspace_dev = NULL (stream-ordered allocation inside the library) and a stream other than the inside pass's give the same
    numbers, bit for bit (every sum has a fixed order)."""
    import torch

    m = I.nn_model()
    d = I.design(5, 0, 40)
    tg, lz, bg, sg, cg = _gpu(B, m, d.aa, d.kind, d.codon_logw, d.pair_logw)
    st = torch.cuda.Stream()
    b2, s2, c2 = tg.marginals(stream=st, own_workspace=False)
    assert (b2.cpu().numpy() == bg).all() and (s2.cpu().numpy() == sg).all() and (c2.cpu().numpy() == cg).all()


def test_marginals_before_inside_rejected(B):
    m = B.Model(I.nn_model())
    tt = B.TensorTrain.build("MW", 0)
    tg, _ = B.inside(m, tt)
    bpp, base, codon = tg.marginals()
    assert abs(float(base.sum()) - 6.0) < 1e-9 and abs(float(codon.sum()) - 2.0) < 1e-9
