"""Pins of the tensor-model oracle (oracle/tensor_model.py) against what the paper and the mathematics fix: explicit
enumeration of sequences x structures with every state contracted as its own tensor diagram (PAPER.md eq S2.1), the
structure counts of eq S2.3 (line 470; tests/golden/structure_counts.txt), the transfer-matrix product of an unpaired strand
(line 448: "q = -log Tr_S[V_0 ... V_{n-1}]", with the tensor train: eq 3.2), and the fixed-sequence reduction."""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from oracle import tensor_model as TM
from paper_2604_19718_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _tt(aa, kind, seed=5):
    tt = O.TT.build(aa, kind, I.codon_logw(seed), I.pair_logw(seed) if kind == I.TT_CODON_PAIR else None)
    return tt.get()


@pytest.mark.parametrize("aa,kind,gamma,xi,mh", [
    ("MF", 0, 2, 2, 3), ("MLF", 0, 2, 2, 3), ("FL", 1, 2, 2, 3), ("LSR", 0, 2, 2, 3), ("LSR", 1, 2, 1, 3), ("RSLG", 0, 2, 2, 3),
    ("LSR", 0, 3, 2, 1), ("SRL", 1, 2, 2, 1), ("GLW", 0, 1, 3, 0), ("MWMW", 0, 3, 2, 1), ("LRSG", 1, 1, 1, 2),
])
def test_recursion_equals_enumeration(aa, kind, gamma, xi, mh):
    """Alg S4.1 with chi-hat (eqs 3.5-3.8) == sum over coding sequences and structures of the state's tensor diagram.  min_hairpin below 3
    makes nested pairs and multi-branch loops reachable at 9-12 nt; a dropped transpose, a swapped B side, a wrong bond index of the
    enclosed block or a missing conformation sum changes the left side only."""
    tm = I.tensor_model(gamma, xi, seed=77 + gamma)
    tm.min_hairpin = mh
    sigma, ops = _tt(aa, kind)
    lz = TM.tm_inside(tm, sigma, ops)
    bf, ns = TM.tm_brute_force(tm, sigma, ops)
    assert ns > 1
    assert abs(lz - bf) <= 1e-12 * max(1.0, abs(bf)), (lz, bf, ns)


def _counts():
    tab = {}
    for line in open(os.path.join(GOLD, "structure_counts.txt")):
        if line.startswith("unlimited"):
            _, n, v = line.split()
            tab[int(n)] = int(v)
    return tab


@pytest.mark.parametrize("n", [5, 12, 20, 24, 30, 36])
def test_unit_model_counts_structures(n):
    """gamma = xi = 1, every entry 1, every two bases may pair, one operator per position: Z = S(n), the number of unpseudoknotted
    structures with hairpins >= 3 (eq S2.3; the tensor model has no interior-loop size limit)."""
    tm = I.tensor_model(1, 1, unit=True)
    ops = [[(0, p % 4, 0, 1.0)] for p in range(n)]
    lz = TM.tm_inside(tm, [1] * (n + 1), ops)
    assert abs(lz - math.log(_counts()[n])) <= 1e-12 * max(1.0, lz)


def test_unit_model_counts_sequences_times_structures():
    """The same with a codon tensor train without weights: Z = prod deg(aa) x S(3L) (line 143)."""
    tm = I.tensor_model(1, 1, unit=True)
    aa = "LSRGMF"
    tt = O.TT.build(aa, I.TT_SINGLE_CODON, None, None)
    sigma, ops = tt.get()
    lz = TM.tm_inside(tm, sigma, ops)
    assert abs(lz - (math.log(6 * 6 * 6 * 4 * 1 * 2) + math.log(_counts()[18]))) <= 1e-12 * lz


@pytest.mark.parametrize("kind", [0, 1])
def test_no_pairs_is_transfer_matrix_product(kind):
    """B = 0: only the unpaired strand remains, Z = sum_{sigma_n} Tr_S of the product of the dressed transfer matrices
    sum_x T_p[x] (x) V[x] (line 448 with the tensor train of eq 3.1)."""
    tm = I.tensor_model(3, 2, seed=11)
    tm.B = np.zeros_like(tm.B)
    sigma, ops = _tt("LSRGAW", kind)
    M = np.eye(3)
    for p, lst in enumerate(ops):
        Tp = np.zeros((3 * sigma[p], 3 * sigma[p + 1]))
        for (a, b, c, x) in lst:
            Tp[a * 3:(a + 1) * 3, c * 3:(c + 1) * 3] += x * tm.V[b]
        M = M @ Tp
    Z = sum(np.trace(tm.S @ M[:, s * 3:(s + 1) * 3]) for s in range(sigma[-1]))
    assert abs(TM.tm_inside(tm, sigma, ops) - math.log(Z)) <= 1e-12 * abs(math.log(Z))


def test_fixed_sequence_reduction():
    """A Met/Trp protein has one coding sequence: log Z(design) = log Z(fixed sequence) + sum of the codon log-weights."""
    tm = I.tensor_model(2, 2, seed=3)
    aa = "MWWMWM"
    cw = I.codon_logw(9)
    tt = O.TT.build(aa, I.TT_SINGLE_CODON, cw, None)
    sigma, ops = tt.get()
    seq = [b for lst in ops for (_, b, _, _) in lst]
    assert len(seq) == 18
    fixed = [[(0, b, 0, 1.0)] for b in seq]
    logw = cw[16 * 0 + 4 * 3 + 2] * aa.count("M") + cw[16 * 3 + 4 * 2 + 2] * aa.count("W")  # AUG, UGG
    assert abs(TM.tm_inside(tm, sigma, ops) - TM.tm_inside(tm, [1] * 19, fixed) - logw) <= 1e-12


def _chi2_states(dist, seqs, pairs):
    """Pearson statistic of sampled (sequence, structure) counts against the exact distribution, states with expected count < 5 pooled."""
    import collections

    J = len(seqs)
    cnt = collections.Counter((tuple(int(v) for v in seqs[k]), tuple(int(v) for v in pairs[k])) for k in range(J))
    assert all(k in dist for k in cnt), "a sampled state lies outside the support"
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
    return chi, len(exp) - 1


@pytest.mark.parametrize("aa,kind,gamma,xi,mh,J,seed", [("LSR", 0, 2, 2, 1, 5000, 1), ("FLM", 1, 2, 1, 0, 4000, 2)])
def test_traceback_samples_the_exact_joint_distribution(aa, kind, gamma, xi, mh, J, seed):
    """tm_sample against the exact distribution over (sequence, structure) from explicit enumeration (thousands of states): every sampled
    state lies in the support and the pooled chi-square stays within 4 standard deviations (a wrong alternative weight, order or child
    element shifts whole families of states); every decision's alternatives sum to the stored block entry it decomposes (1e-12)."""
    tm = I.tensor_model(gamma, xi, seed=79)
    tm.min_hairpin = mh
    sigma, ops = _tt(aa, kind)
    _, Q = TM.tm_inside(tm, sigma, ops, return_Q=True)
    worst = [0.0]
    orig = TM._pick

    def checked(alts, total, u):
        worst[0] = max(worst[0], abs(sum(w for _, w in alts if w > 0.0) - total) / total)
        return orig(alts, total, u)

    TM._pick = checked
    try:
        seqs, pairs = TM.tm_sample(tm, sigma, ops, Q, J, seed, O.uniform)
    finally:
        TM._pick = orig
    assert worst[0] <= 1e-12
    chi, dof = _chi2_states(TM.tm_state_distribution(tm, sigma, ops), seqs, pairs)
    assert abs(chi - dof) <= 4.0 * math.sqrt(2.0 * dof), (chi, dof)
    # the sampled sequences code for the protein: every codon of the sample translates to its residue
    code = "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF"  # index 16 b0 + 4 b1 + b2, A C G U
    for k in range(0, J, 97):
        assert "".join(code[16 * seqs[k][3 * r] + 4 * seqs[k][3 * r + 1] + seqs[k][3 * r + 2]] for r in range(len(aa))) == aa
