"""GPU parity of the tensor-model recursion (cdz_tm_inside; eqs 3.5-3.8) against oracle/tensor_model.py, through the
C ABI: every block of Q (upper Q_{i,j} and lower Q_{j,i}) element by element, log Z at 1e-9 relative (DESIGN.md c-13), the closed forms of
the oracle's pins at sizes the oracle cannot reach, and the edge cases."""
import math
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding

    binding.lib()
    return binding


@pytest.fixture(scope="module")
def I():
    from paper_2604_19718_b200 import inputs

    return inputs


def _both(B, I, aa, kind, seed=5):
    from oracle import oracle as O

    cw, pw = I.codon_logw(seed), (I.pair_logw(seed) if kind == I.TT_CODON_PAIR else None)
    return B.TensorTrain.build(aa, kind, cw, pw), O.TT.build(aa, kind, cw, pw).get()


@pytest.mark.parametrize("cfg,L,gamma,xi,mh", [
    (1, 4, 2, 2, 3), (1, 20, 2, 2, 3), (1, 20, 4, 2, 3), (5, 12, 2, 2, 3), (5, 12, 4, 1, 1), (1, 30, 3, 3, 0), (2, 25, 2, 2, 3),
    (1, 40, 8, 1, 3),
])
def test_blocks_and_logz_vs_oracle(B, I, cfg, L, gamma, xi, mh):
    """Every stored block against the plain Alg S4.1 of the oracle: several 64-blocks (GEMM tiles, split-K, in-block edges of both kinds),
    both tensor trains, gamma 2..8, ragged last block."""
    from oracle import tensor_model as TM

    d = I.design(cfg, 0, L)
    tm = I.tensor_model(gamma, xi, seed=100 + gamma)
    tm.min_hairpin = mh
    tg, (sigma, ops) = _both(B, I, d.aa, d.kind, d.seed)
    lz_o, Q = TM.tm_inside(tm, sigma, ops, return_Q=True)
    run = B.TensorModelPass(tm, tg)
    assert abs(run.logZ - lz_o) <= 1e-9 * abs(lz_o), (run.logZ, lz_o)
    n = len(ops)
    worst = 0.0
    for i in range(n + 1):
        for j in range(i, n + 1):
            v, sh = run.block(0, i, j)
            ref = Q[i][j].reshape(-1)
            got = v * 2.0 ** sh
            worst = max(worst, float(np.max(np.abs(got - ref) / (np.abs(ref) + 1e-300 + 1e-13 * np.max(np.abs(ref))))))
            if j > i:
                v, sh = run.block(1, i, j)
                ref = Q[j][i].reshape(-1)
                got = v * 2.0 ** sh
                worst = max(worst, float(np.max(np.abs(got - ref) / (np.abs(ref) + 1e-300 + 1e-13 * max(1e-300, np.max(np.abs(ref)))))))
    assert worst <= 1e-10, worst


def _counts():
    tab = {}
    for line in open(os.path.join(GOLD, "structure_counts.txt")):
        if line.startswith("unlimited"):
            _, n, v = line.split()
            tab[int(n)] = int(v)
    return tab


@pytest.mark.parametrize("n", [5, 20, 37, 38])
def test_unit_model_structure_counts(B, I, n):
    """gamma = xi = 1, all ones, every two bases pair, one operator per position: Z = S(n) of eq S2.3 (tests/golden/structure_counts.txt)."""
    tm = I.tensor_model(1, 1, unit=True)
    tg = B.TensorTrain.from_operators([[(0, p % 4, 0, 1.0)] for p in range(n)])
    run = B.TensorModelPass(tm, tg)
    assert abs(run.logZ - math.log(_counts()[n])) <= 1e-12 * run.logZ


def _log_structure_count(n, mh=3):
    """log S(n) by the scalar recursion S(m) = S(m-1) + sum_k S(k) S(m-2-k), hairpins >= mh (eq S2.3), in exact integers."""
    S = [1] * (n + 1)
    for m in range(1, n + 1):
        v = S[m - 1]
        for k in range(0, m - 1):  # first base paired with k+1 ... enclosed k bases, rest m-2-k
            if k >= mh:
                v += S[k] * S[m - 2 - k]
        S[m] = v
    return math.log(S[n])


def test_unit_model_large_closed_form(B, I):
    """2400 nt with a weightless single-codon tensor train (60+ blocks, split-K, the pilot scale in use): log Z = sum log deg + log S(n),
    S(n) in exact integer arithmetic -- nothing of the recursion under test is used on the right-hand side."""
    tm = I.tensor_model(1, 1, unit=True)
    aa = I.protein(777, 800)
    deg = {"A": 4, "C": 2, "D": 2, "E": 2, "F": 2, "G": 4, "H": 2, "I": 3, "K": 2, "L": 6, "M": 1, "N": 2, "P": 4, "Q": 2, "R": 6, "S": 6,
           "T": 4, "V": 4, "W": 1, "Y": 2}
    tg = B.TensorTrain.build(aa, I.TT_SINGLE_CODON, None, None)
    run = B.TensorModelPass(tm, tg)
    ref = sum(math.log(deg[a]) for a in aa) + _log_structure_count(3 * len(aa))
    assert run.info.NB >= 50 and run.info.scale_rate != 0.0
    assert abs(run.logZ - ref) <= 1e-9 * ref, (run.logZ, ref)


def test_no_pairs_transfer_product_and_determinism(B, I):
    """B = 0 at 900 nt: Z = sum_{sigma_n} Tr_S of the product of the dressed transfer matrices (line 448), accumulated here in log space."""
    tm = I.tensor_model(3, 2, seed=11)
    tm.B = np.zeros_like(tm.B)
    d = I.design(2, 0, 300)
    tg, (sigma, ops) = _both(B, I, d.aa, d.kind, d.seed)
    M, logs = np.eye(3), 0.0
    for p, lst in enumerate(ops):
        Tp = np.zeros((3 * sigma[p], 3 * sigma[p + 1]))
        for (a, b, c, x) in lst:
            Tp[a * 3:(a + 1) * 3, c * 3:(c + 1) * 3] += x * tm.V[b]
        M = M @ Tp
        s = M.max()
        M, logs = M / s, logs + math.log(s)
    ref = math.log(sum(np.trace(tm.S @ M[:, s * 3:(s + 1) * 3]) for s in range(sigma[-1]))) + logs
    run = B.TensorModelPass(tm, tg)
    assert abs(run.logZ - ref) <= 1e-9 * abs(ref), (run.logZ, ref)
    first = run.logZ
    assert run.rerun() == first


def test_prefix_chain_config2(B, I):
    """Config-2 design (300 aa, codon-pair tensor train, gamma 4, xi 2) at full size: finite, deterministic, and the blocks of its first
    36 nt equal the oracle's run on that prefix (Q_{i,j} depends on positions i..j-1 only), the uniform scale undone."""
    from oracle import oracle as O
    from oracle import tensor_model as TM

    d = I.design(2, 0)
    tm = I.tensor_model(4, 2)
    tg = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    run = B.TensorModelPass(tm, tg)
    assert math.isfinite(run.logZ) and run.info.scale_rate != 0.0
    sigma, ops = O.TT.build(d.aa[:12], d.kind, d.codon_logw, d.pair_logw).get()
    _, Q = TM.tm_inside(tm, sigma, ops, return_Q=True)
    for (i, j) in ((0, 36), (0, 20), (7, 33), (3, 4), (12, 35)):
        if j == 36:
            continue  # the last bond of the prefix train is not the bond of the full train at that point
        v, sh = run.block(0, i, j)
        ref = Q[i][j].reshape(-1)
        assert np.allclose(v * 2.0 ** sh, ref, rtol=1e-10, atol=0.0), (i, j)
        v, sh = run.block(1, i, j)
        assert np.allclose(v * 2.0 ** sh, Q[j][i].reshape(-1), rtol=1e-10, atol=1e-300), (i, j)


def test_errors(B, I):
    tm = I.tensor_model(2, 2)
    tg = B.TensorTrain.build("MF", I.TT_SINGLE_CODON, None, None)
    bad = I.tensor_model(2, 2)
    bad.V = -bad.V
    with pytest.raises(B.CdzError):
        B.TensorModelPass(bad, tg)
    big = I.tensor_model(2, 2)
    big.gamma = 9
    with pytest.raises(B.CdzError):
        B.TensorModelPass(big, tg)
    assert math.isfinite(B.TensorModelPass(tm, tg).logZ)


CODE = "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF"  # index 16 b0 + 4 b1 + b2 over A C G U


def _valid_state(aa, seq, pair, mh):
    n = len(seq)
    assert "".join(CODE[16 * seq[3 * r] + 4 * seq[3 * r + 1] + seq[3 * r + 2]] for r in range(len(aa))) == aa
    can = {(0, 3), (3, 0), (1, 2), (2, 1), (2, 3), (3, 2)}
    stack = []
    for i in range(n):
        jn = int(pair[i])
        if jn < 0:
            continue
        assert int(pair[jn]) == i
        if jn > i:
            assert jn - i - 1 >= mh and (int(seq[i]), int(seq[jn])) in can
            stack.append(jn)
        else:
            assert stack and stack.pop() == i  # non-crossing


@pytest.mark.parametrize("cfg,L,gamma,xi,mh,J", [(1, 20, 2, 2, 3, 100), (1, 12, 3, 1, 0, 100), (5, 6, 2, 2, 1, 40), (1, 30, 4, 2, 3, 40)])
def test_tm_samples_bit_exact(B, I, cfg, L, gamma, xi, mh, J):
    """cdz_tm_sample == the oracle's traceback for the same seed: every nucleotide and every partner of every sample."""
    from oracle import oracle as O
    from oracle import tensor_model as TM

    d = I.design(cfg, 0, L)
    tm = I.tensor_model(gamma, xi, seed=100 + gamma)
    tm.min_hairpin = mh
    tg, (sigma, ops) = _both(B, I, d.aa, d.kind, d.seed)
    _, Q = TM.tm_inside(tm, sigma, ops, return_Q=True)
    so, po = TM.tm_sample(tm, sigma, ops, Q, J, d.sample_seed, O.uniform)
    run = B.TensorModelPass(tm, tg)
    sg, pg = run.sample(J, d.sample_seed)
    assert (sg.cpu().numpy() == so).all() and (pg.cpu().numpy() == po).all()
    for k in range(0, J, 7):
        _valid_state(d.aa, so[k], po[k], mh)


def test_tm_samples_follow_the_exact_distribution(B, I):
    """40000 GPU samples of a 9-nt design against the exact (sequence, structure) distribution from enumeration (oracle): support and
    pooled chi-square within 4 standard deviations."""
    import collections

    from oracle import oracle as O
    from oracle import tensor_model as TM

    tm = I.tensor_model(2, 2, seed=79)
    tm.min_hairpin = 1
    cw = I.codon_logw(5)
    tg = B.TensorTrain.build("LSR", I.TT_SINGLE_CODON, cw, None)
    sigma, ops = O.TT.build("LSR", I.TT_SINGLE_CODON, cw, None).get()
    dist = TM.tm_state_distribution(tm, sigma, ops)
    J = 40000
    run = B.TensorModelPass(tm, tg)
    sg, pg = run.sample(J, 4242)
    sg, pg = sg.cpu().numpy(), pg.cpu().numpy()
    cnt = collections.Counter((tuple(int(v) for v in sg[k]), tuple(int(v) for v in pg[k])) for k in range(J))
    assert all(k in dist for k in cnt)
    exp, obs, pe, po = [], [], 0.0, 0.0
    for k, p in sorted(dist.items(), key=lambda kv: -kv[1]):
        e, o = p * J, cnt.get(k, 0)
        if e >= 5:
            exp.append(e)
            obs.append(o)
        else:
            pe += e
            po += o
    if pe > 0:
        exp.append(pe)
        obs.append(po)
    chi = sum((o - e) ** 2 / e for o, e in zip(obs, exp))
    dof = len(exp) - 1
    assert abs(chi - dof) <= 4.0 * math.sqrt(2.0 * dof), (chi, dof)


def test_tm_samples_full_size_valid_and_deterministic(B, I):
    """Config-2 design (900 nt, codon-pair train, gamma 4, xi 2): 64 samples are coding sequences of the protein with unpseudoknotted
    structures of canonical pairs and hairpins >= 3; the same seed gives the same samples."""
    d = I.design(2, 0)
    tm = I.tensor_model(4, 2)
    tg = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    run = B.TensorModelPass(tm, tg)
    s1, p1 = run.sample(64, 99)
    s2, p2 = run.sample(64, 99)
    assert (s1 == s2).all() and (p1 == p2).all()
    s1, p1 = s1.cpu().numpy(), p1.cpu().numpy()
    for k in range(64):
        _valid_state(d.aa, s1[k], p1[k], 3)
    assert (p1 >= 0).sum() > 0


def test_generic_operator_list_bond_dimension_8(B, I):
    """Generic operator list of bond dimension 8 with gamma = 4: 32-dimensional boundary points (the kernel limit), two points per 64-block,
    so nearly every k-sum crosses blocks; every block of Q and 8 samples against the oracle."""
    from oracle import oracle as O
    from oracle import tensor_model as TM

    ops = I.closed_form_inputs("zero8", 30)
    tm = I.tensor_model(4, 2, seed=17)
    tg = B.TensorTrain.from_operators(ops)
    sigma, oo = O.TT.from_ops(ops).get()
    lz_o, Q = TM.tm_inside(tm, sigma, oo, return_Q=True)
    run = B.TensorModelPass(tm, tg)
    assert run.info.NB >= 12
    assert abs(run.logZ - lz_o) <= 1e-9 * abs(lz_o)
    n = len(ops)
    for i in range(0, n + 1, 3):
        for j in range(i, n + 1):
            v, sh = run.block(0, i, j)
            ref = Q[i][j].reshape(-1)
            assert np.allclose(v * 2.0 ** sh, ref, rtol=1e-10, atol=1e-13 * max(1e-300, np.abs(ref).max())), (i, j)
    so, po = TM.tm_sample(tm, sigma, oo, Q, 8, 5, O.uniform)
    sg, pg = run.sample(8, 5)
    assert (sg.cpu().numpy() == so).all() and (pg.cpu().numpy() == po).all()


def test_tiny_and_limits(B, I):
    """One residue (3 nt, no pair possible), xi = 4, gamma = 8 with a bond-4 train (32-dimensional points), and the rejected sizes."""
    from oracle import oracle as O
    from oracle import tensor_model as TM

    for aa, gamma, xi in (("M", 2, 2), ("L", 3, 4), ("LSRW", 8, 1)):
        tm = I.tensor_model(gamma, xi, seed=5)
        tm.min_hairpin = 1
        tg = B.TensorTrain.build(aa, I.TT_SINGLE_CODON, None, None)
        sigma, ops = O.TT.build(aa, I.TT_SINGLE_CODON, None, None).get()
        lz = TM.tm_inside(tm, sigma, ops)
        assert abs(B.TensorModelPass(tm, tg).logZ - lz) <= 1e-9 * max(1.0, abs(lz))
    # gamma x bond > 32 is rejected: gamma 8 with a codon-pair train (bond 6)
    tg = B.TensorTrain.build("LSR", I.TT_CODON_PAIR, None, None)
    with pytest.raises(B.CdzError):
        B.TensorModelPass(I.tensor_model(8, 1), tg)
