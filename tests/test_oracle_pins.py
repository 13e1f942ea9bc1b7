"""Pins of the CPU oracle against things other than itself (CPU only).

Each test names what fixes the expected value: a closed form, brute-force enumeration of the plain
definition, a reduction to a textbook routine, or a value printed in SURVEY.md App. B/C by the
surveyor's independent prototype (tests/golden/README.md).
"""
import copy
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2604_19718_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")
DEG = {a: "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF".count(a) for a in I.AMINO}


def rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def build(aa, kind, cw, pw):
    return O.TT.build(aa, kind, I.tm1_codon_logw() if cw else None, I.tm1_pair_logw() if pw else None)


# ---------------------------------------------------------------- generator
def test_generator_check_values():
    """SURVEY.md App. C 'generator check values'."""
    m = I.nn_model()
    np.testing.assert_allclose(m.stack[0], [-2.371228, -3.069518, -1.319718, -3.327908, -2.674364, -3.254276], atol=6e-7)
    assert abs(m.stack[5, 5] - -2.483470) < 6e-7
    assert abs(m.tmm[0, 0, 0] - -1.412304) < 6e-7 and abs(m.tmm[5, 3, 3] - -0.831109) < 6e-7
    np.testing.assert_allclose(I.codon_logw(1000)[:3], [-0.237386, -0.397274, -0.617901], atol=6e-7)
    assert abs(I.pair_logw(1000)[0, 0] - 0.085029) < 6e-7
    for p in range(6):  # "symmetric under pair reversal" (BASELINE.json configs[0])
        for q in range(6):
            assert m.stack[p, q] == m.stack[I.REV_PAIR[q], I.REV_PAIR[p]]
    assert abs(m.kT - 0.6163314008) < 1e-9


def test_protein_stream_prefix_stable():
    assert I.protein(1000, 20) == "PPTWVRLATTIWWMTFILCS"
    assert I.protein(1000, 50)[:20] == I.protein(1000, 20)


# ---------------------------------------------------------------- tensor train
@pytest.mark.parametrize("aa", ["MW", "RSLG", "LSRGAVI", I.protein(1000, 20), I.AMINO])
@pytest.mark.parametrize("kind", [0, 1])
def test_tt_counts_sequences(aa, kind):
    """Unweighted TT: q_seq = -log |Phi(psi)| = prod of codon degeneracies."""
    tt = O.TT.build(aa, kind)
    want = sum(math.log(DEG[a]) for a in aa)
    assert abs(tt.logsum() - want) < 1e-12


def test_tt_bond_dimensions():
    """Sigma-bar of SURVEY.md App. C (single: 1/#first/#third bases; pair: deg(prev), deg, deg)."""
    for cfg, L, aa, sbar, _ in rows("appendix_c.txt"):
        d = I.design(int(cfg), 0, int(L))
        assert d.aa == aa
        sig, ops = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw).get()
        assert sum(sig[:-1]) == int(sbar)
        assert sig[0] == 1


def test_tt_weight_sum_direct_enumeration():
    """sum_phi W(phi) from the TT (eq 3.2) equals direct enumeration over codon choices."""
    code = "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF"
    cw, pw = I.tm1_codon_logw(), I.tm1_pair_logw()
    aa = "RSLG"
    cods = [[c for c in range(64) if code[c] == a] for a in aa]
    import itertools

    tot1 = tot2 = 0.0
    for choice in itertools.product(*cods):
        w1 = sum(cw[c] for c in choice)
        w2 = w1 + sum(pw[choice[k - 1], choice[k]] for k in range(1, len(choice)))
        tot1 += math.exp(w1)
        tot2 += math.exp(w2)
    assert abs(O.TT.build(aa, 0, cw).logsum() - math.log(tot1)) < 1e-12
    assert abs(O.TT.build(aa, 1, cw, pw).logsum() - math.log(tot2)) < 1e-12
    # SURVEY.md section 8(c) prints both numbers
    assert abs(math.log(tot1) - 6.717883310603) < 1e-11
    assert abs(math.log(tot2) - 6.740724276906) < 1e-11


def test_codon_weight_shift():
    """Adding delta to every codon log-weight of one amino acid shifts log Z by delta per occurrence (line 157)."""
    m = I.tm1_model()
    cw = I.tm1_codon_logw()
    cw2 = cw.copy()
    code = "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF"
    for c in range(64):
        if code[c] == "S":
            cw2[c] += 0.37
    a = O.inside(m, O.TT.build("RSLGS", 0, cw)).logZ
    b = O.inside(m, O.TT.build("RSLGS", 0, cw2)).logZ
    assert abs(b - a - 2 * 0.37) < 1e-12


# ---------------------------------------------------------------- structure enumeration
def S_closed(nmax):
    """PAPER.md eq S2.3 (line 470) with hairpins >= 3 (line 483): S(n)=S(n-1)+sum_k S(k)S(n-2-k), n-2-k>=3."""
    S = [1] * (nmax + 1)
    for n in range(1, nmax + 1):
        S[n] = S[n - 1] + sum(S[k] * S[n - 2 - k] for k in range(0, n - 1) if n - 2 - k >= 3)
    return S


def test_structure_counts_enumeration_vs_recursion():
    S = S_closed(20)
    for kind, n, val in rows("structure_counts.txt"):
        n, val = int(n), int(val)
        if kind == "unlimited" and n <= 20:
            assert S[n] == val
            if n >= 1 and n <= 16:
                assert O.count_structures(n) == val  # brute-force enumerator of the oracle


def test_zero_energy_dp_counts():
    """Zero-energy all-pairs model: Z = #Phi x S(n) (BASELINE.json north_star closed form)."""
    m = I.zero_energy_model()
    tab = {(k, int(n)): int(v) for k, n, v in rows("structure_counts.txt")}
    for n in (12, 24, 30, 36, 37):
        tt = O.TT.from_ops([[(0, 0, 0, 1.0)]] * n)
        z = math.exp(O.inside(m, tt).logZ)
        assert abs(z / tab[("unlimited", n)] - 1) < 1e-14
    for n in (38, 39, 40, 50, 60):  # interior loops limited to 30 unpaired: first differs at n=38
        tt = O.TT.from_ops([[(0, 0, 0, 1.0)]] * n)
        z = math.exp(O.inside(m, tt).logZ)
        assert abs(z / tab[("limit30", n)] - 1) < 1e-14
    S = S_closed(15)
    for aa, want in (("LSR", 6912), ("RSLG", 236736), ("GAVLI", 2858112)):
        tt = O.TT.build(aa, 0)
        nseq = math.prod(DEG[a] for a in aa)
        assert want == nseq * S[3 * len(aa)]
        assert abs(math.exp(O.inside(m, tt).logZ) / want - 1) < 1e-14
        assert abs(math.exp(O.inside(m, O.TT.build(aa, 1)).logZ) / want - 1) < 1e-14


def test_zero_energy_canonical_pairs():
    """canonical pairs only, zero energy: Z = 2516 (LSR), 46774 (RSLG)."""
    m = I.zero_energy_model(allow_all_pairs=0)
    for aa, want in (("LSR", 2516), ("RSLG", 46774)):
        tt = O.TT.build(aa, 0)
        assert abs(math.exp(O.inside(m, tt).logZ) - want) < 1e-8
        bf = O.brute_force(m, tt)
        assert abs(math.exp(bf["logZ"]) - want) < 1e-8 and bf["n_states"] == want


# ---------------------------------------------------------------- energy evaluator, by hand
def test_energy_hand_cases():
    m = I.nn_model()
    kT = m.kT
    A, Cc, G, U = 0, 1, 2, 3
    # hairpin GAAAC closed by G-C (type 2), loop AAA: H(3) + tmm[2][A][A]
    seq = [G, A, A, A, Cc]
    e, ok = O.energy(m, seq, [4, -1, -1, -1, 0])
    assert ok and abs(e - (5.4 + 1.75 * kT * math.log(3 / 9) + m.tmm[2, A, A])) < 1e-12
    # too-short hairpin is not a structure
    assert not O.energy(m, [G, A, A, Cc], [3, -1, -1, 0])[1]
    # non-pairable
    assert not O.energy(m, [A, A, A, A, A], [4, -1, -1, -1, 0])[1]
    # stack: GG AAA CC -> (0,6) G-C type 2 closing, (1,5) G-C type 2 inner
    seq = [G, G, A, A, A, Cc, Cc]
    e, ok = O.energy(m, seq, [6, 5, -1, -1, -1, 1, 0])
    assert ok and abs(e - (m.stack[2, 2] + 5.4 + 1.75 * kT * math.log(3 / 9) + m.tmm[2, A, A])) < 1e-12
    # bulge of 1 on the left: G A G AAA C C : (0,7),(2,6)
    seq = [G, A, G, A, A, A, Cc, Cc]
    e, ok = O.energy(m, seq, [7, -1, 6, -1, -1, -1, 2, 0])
    hp = 5.4 + 1.75 * kT * math.log(3 / 9) + m.tmm[2, A, A]
    assert ok and abs(e - (3.8 + m.stack[2, 2] + hp)) < 1e-12
    # bulge of 2 on the right: G G AAA C UU C -> (0,8),(1,5)
    seq = [G, G, A, A, A, Cc, U, U, Cc]
    e, ok = O.energy(m, seq, [8, 5, -1, -1, -1, 1, -1, -1, 0])
    assert ok and abs(e - (3.8 + 1.75 * kT * math.log(2) + hp)) < 1e-12
    # 1x2 interior: G A G AAA C UC C : closing (0,9) G-C, inner (2,6) G-C; mismatches:
    #   closing tmm[p(G,C)][phi_1=A][phi_8=C]; inner pair read as (phi_l,phi_k)=(C,G) type 1 with phi_{l+1}=U, phi_{k-1}=A
    seq = [G, A, G, A, A, A, Cc, U, Cc, Cc]
    e, ok = O.energy(m, seq, [9, -1, 6, -1, -1, -1, 2, -1, -1, 0])
    want = 2.0 + 1.75 * kT * math.log(3 / 2) + m.tmm[2, A, Cc] + m.tmm[1, U, A] + hp
    assert ok and abs(e - want) < 1e-12
    # multiloop with 2 branches, 1 unpaired: G [GAAAC] A [GAAAC] C
    seq = [G] + [G, A, A, A, Cc] + [A] + [G, A, A, A, Cc] + [Cc]
    pair = [12, 5, -1, -1, -1, 1, -1, 11, -1, -1, -1, 7, 0]
    e, ok = O.energy(m, seq, pair)
    assert ok and abs(e - (3.4 + 0.4 * 3 + 0.0 * 1 + 2 * hp)) < 1e-12
    # exterior loop costs nothing; crossing pairs rejected
    assert O.energy(m, [A] * 5, [-1] * 5) == (0.0, True)
    assert not O.energy(m, [G, G, A, A, A, Cc, Cc, A, A], [5, 6, -1, -1, -1, 0, 1, -1, -1])[1]
    # interior loop limit 30 (BASELINE.json configs[0])
    seq = [G] + [A] * 16 + [G, A, A, A, Cc] + [A] * 15 + [Cc]
    pair = [-1] * len(seq)
    pair[0], pair[len(seq) - 1] = len(seq) - 1, 0
    pair[17], pair[21] = 21, 17
    assert not O.energy(m, seq, pair)[1]
    seq2 = seq[:16] + seq[17:]
    pair2 = [-1] * len(seq2)
    pair2[0], pair2[len(seq2) - 1] = len(seq2) - 1, 0
    pair2[16], pair2[20] = 20, 16
    assert O.energy(m, seq2, pair2)[1]


# ---------------------------------------------------------------- inside recursion
@pytest.mark.parametrize("row", rows("appendix_b.txt"), ids=lambda r: "-".join(r[:5]))
def test_appendix_b(row):
    """SURVEY.md App. B pinned log Z (independent prototype) and brute force == DP."""
    aa, kind, cw, pw, mi, ref = row[0], int(row[1]), int(row[2]), int(row[3]), int(row[4]), float(row[5])
    m = I.tm1_model()
    m.max_interior = mi
    tt = build(aa, kind, cw, pw)
    bf = O.brute_force(m, tt)
    dp = O.inside(m, tt)
    assert abs(bf["logZ"] - ref) < 2e-12
    assert abs(dp.logZ - bf["logZ"]) < 5e-14 * max(1.0, abs(ref))


@pytest.mark.parametrize("seed", range(8))
def test_inside_vs_brute_force_random(seed):
    """Random small proteins, BJ generator and model: DP == enumeration of eqs 2.1-2.4."""
    m = I.nn_model(19718 + seed)
    L = 3 + seed % 2
    aa = I.protein(77 + seed, L)
    kind = seed % 2
    tt = O.TT.build(aa, kind, I.codon_logw(seed), I.pair_logw(seed) if kind else None)
    bf = O.brute_force(m, tt)
    dp = O.inside(m, tt)
    assert abs(dp.logZ - bf["logZ"]) < 1e-13 * max(1.0, abs(bf["logZ"]))


def test_appendix_c_logz():
    m = I.nn_model()
    for cfg, L, aa, sbar, ref in rows("appendix_c.txt"):
        d = I.design(int(cfg), 0, int(L))
        tt = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
        assert abs(O.inside(m, tt).logZ - float(ref)) < 2e-12 * float(ref)


@pytest.mark.parametrize("aa", ["MWMWMW", "WMMWWMWMMMWWMWMWMMWW"])
def test_single_codon_protein_reduces_to_mccaskill(aa):
    """Met/Trp-only protein: one sequence, so log Z = scalar McCaskill + log W (BJ north_star invariant)."""
    for m in (I.tm1_model(), I.nn_model()):
        cw = I.tm1_codon_logw()
        code = {"M": (0, 3, 2), "W": (3, 2, 2)}
        seq = [b for a in aa for b in code[a]]
        logW = sum(cw[16 * code[a][0] + 4 * code[a][1] + code[a][2]] for a in aa)
        want = O.mccaskill(m, seq) + logW
        for kind in (0, 1):
            got = O.inside(m, O.TT.build(aa, kind, cw, I.tm1_pair_logw() * 0 if kind else None)).logZ
            assert abs(got - want) < 1e-13 * max(1.0, abs(want))


def test_mccaskill_vs_enumeration():
    """The textbook scalar routine itself, against brute force over structures of a fixed sequence."""
    m = I.nn_model()
    g = I.SplitMix64(5)
    for n in (8, 13, 17):
        seq = [int(4 * g.uniform()) for _ in range(n)]
        tt = O.TT.from_ops([[(0, b, 0, 1.0)] for b in seq])
        assert abs(O.mccaskill(m, seq) - O.brute_force(m, tt)["logZ"]) < 1e-13


def test_noncoding_operator_lists():
    """Generic operator lists: free nucleotides with bonuses; DP == brute force."""
    m = I.tm1_model()
    ops = [[(0, b, 0, 1.0 + 0.1 * b + 0.01 * i) for b in range(4)] for i in range(8)]
    tt = O.TT.from_ops(ops)
    assert abs(O.inside(m, tt).logZ - O.brute_force(m, tt)["logZ"]) < 1e-13


def test_short_cells_empty():
    """B_{i,j} = 0 for |j-i| < 4."""
    m = I.tm1_model()
    t = O.inside(m, build("RSLG", 0, 1, 0))
    for i in range(12):
        for j in range(i, min(12, i + 4)):
            assert not t.cell(0, i, j).any()


# ---------------------------------------------------------------- brute-force marginals (definition level)
def test_rslg_marginals_brute_force_golden():
    m = I.tm1_model()
    bf = O.brute_force(m, build("RSLG", 0, 1, 0), marginals=True)
    idx = {c: k for k, c in enumerate("ACGU")}
    for r in rows("rslg_marginals.txt"):
        if r[0] == "punp":
            np.testing.assert_allclose(np.diag(bf["bpp"]), [float(v) for v in r[1:]], atol=6e-10)
        elif r[0] == "pair":
            assert abs(bf["bpp"][int(r[1]), int(r[2])] - float(r[3])) < 6e-10
        else:
            c = 16 * idx[r[2][0]] + 4 * idx[r[2][1]] + idx[r[2][2]]
            assert abs(bf["codon"][int(r[1]), c] - float(r[3])) < 6e-10
    # doubly stochastic including the diagonal
    P = np.triu(bf["bpp"], 1)
    np.testing.assert_allclose((P + P.T).sum(1) + np.diag(bf["bpp"]), 1.0, atol=1e-12)
    np.testing.assert_allclose(bf["codon"].sum(1), 1.0, atol=1e-12)
    np.testing.assert_allclose(bf["base"].sum(1), 1.0, atol=1e-12)


# ---------------------------------------------------------------- sampler
def _chi2_pvalue(stat, dof):
    from scipy.stats import chi2

    return float(chi2.sf(stat, dof))


@pytest.mark.parametrize("aa,kind", [("LSR", 0), ("RSLG", 0), ("LSR", 1), ("MFL", 1)])
def test_sampler_exact_joint_distribution(aa, kind):
    """Samples (phi,s) follow p = W e^{-E/kT}/Z exactly: chi-square over the joint support (n <= 12)."""
    m = I.tm1_model()
    m.ml_a = 0.4  # make multiloops / rarer states visible
    tt = build(aa, kind, 1, kind)
    t = O.inside(m, tt)
    J = 40000
    seq, pair = t.sample(J, 12345)
    seq2, pair2 = t.sample(J, 12345)
    assert (seq == seq2).all() and (pair == pair2).all()  # determinism
    from collections import Counter

    cnt = Counter((s.tobytes(), p.tobytes()) for s, p in zip(seq, pair))
    stat, dof, seen_p, seen_n = 0.0, 0, 0.0, 0
    pool_e = pool_o = 0.0
    for (sb, pb), c in cnt.items():
        s = np.frombuffer(sb, dtype=np.uint8)
        p = np.frombuffer(pb, dtype=np.int32)
        lw = O.logweight(m, tt, s, p)
        assert np.isfinite(lw), "sampled an invalid state"
        pr = math.exp(lw - t.logZ)
        seen_p += pr
        seen_n += c
        e = J * pr
        if e >= 10:
            stat += (c - e) ** 2 / e
            dof += 1
        else:
            pool_e += e
            pool_o += c
    pool_e += J * max(0.0, 1.0 - seen_p)  # unseen states
    if pool_e >= 10:
        stat += (pool_o - pool_e) ** 2 / pool_e
        dof += 1
    assert dof > 5
    assert _chi2_pvalue(stat, dof - 1) > 1e-3


def test_sampler_marginals_chi2_config1_prefix():
    """Sample frequencies vs exact (brute-force) codon marginals on a 4-aa prefix of BJ config 1."""
    m = I.nn_model()
    d = I.design(1, 0, 4)
    tt = O.TT.build(d.aa, d.kind, d.codon_logw)
    bf = O.brute_force(m, tt, marginals=True)
    t = O.inside(m, tt)
    J = 20000
    seq, pair = t.sample(J, d.sample_seed)
    stat, dof = 0.0, 0
    for k in range(len(d.aa)):
        cod = 16 * seq[:, 3 * k].astype(int) + 4 * seq[:, 3 * k + 1] + seq[:, 3 * k + 2]
        obs = np.bincount(cod, minlength=64)
        assert obs[bf["codon"][k] == 0].sum() == 0  # zero mass on disallowed codons
        e = J * bf["codon"][k]
        big = e >= 5
        if big.sum() >= 2:
            stat += ((obs[big] - e[big]) ** 2 / e[big]).sum()
            dof += big.sum() - 1
    unp = (pair < 0).mean(0)
    np.testing.assert_allclose(unp, np.diag(bf["bpp"]), atol=5 * 0.5 / math.sqrt(J))
    assert _chi2_pvalue(stat, dof) > 1e-3


# ---------------------------------------------------------------- marginals by constrained inside passes
@pytest.mark.parametrize("aa,kind,cw,pw", [("RSLG", 0, 1, 0), ("LSR", 1, 1, 1), ("MFL", 1, 1, 1), ("GRL", 0, 0, 0)])
def test_marginals_equal_brute_force(aa, kind, cw, pw):
    """orc_marginals (eqs 2.5-2.7 as ratios of restricted partition functions) against explicit enumeration of every
    (sequence, structure): base-pair matrix, base marginals, codon marginals."""
    m = I.tm1_model()
    tt = build(aa, kind, cw, pw)
    bf = O.brute_force(m, tt, marginals=True)
    bpp, base, codon = O.inside(m, tt).marginals()
    np.testing.assert_allclose(bpp, bf["bpp"], atol=1e-12)
    np.testing.assert_allclose(base, bf["base"], atol=1e-12)
    np.testing.assert_allclose(codon, bf["codon"], atol=1e-12)


def test_marginals_sum_rules_24nt():
    """Beyond brute force (n = 24): rows of the pair matrix + unpaired probability sum to 1, base and codon
    marginals are normalised, foreign codons carry zero mass, base marginals are the codon marginals summed per nucleotide."""
    m = I.nn_model()
    d = I.design(1, 0, 8)
    tt = O.TT.build(d.aa, d.kind, d.codon_logw)
    bpp, base, codon = O.inside(m, tt).marginals()
    P = np.triu(bpp, 1)
    np.testing.assert_allclose((P + P.T).sum(1) + np.diag(bpp), 1.0, atol=1e-12)
    assert (np.diag(bpp) >= -1e-15).all() and (P >= 0).all()
    np.testing.assert_allclose(base.sum(1), 1.0, atol=1e-12)
    np.testing.assert_allclose(codon.sum(1), 1.0, atol=1e-12)
    code = "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF"
    for k, a in enumerate(d.aa):
        foreign = np.array([code[c] != a for c in range(64)])
        assert codon[k][foreign].sum() == 0.0
        for pos in range(3):
            for b in range(4):
                sel = np.array([((c >> (2 * (2 - pos))) & 3) == b for c in range(64)])
                assert abs(codon[k][sel].sum() - base[3 * k + pos, b]) < 1e-12


# ---------------------------------------------------------------- decision uniforms, per-position codon weights
def test_uniform_hash_known_answers():
    """orc_uniform (SURVEY App. C "decision uniforms") against things other than itself: (a) its first round with seed 0 and
    v = 0 is SplitMix64's first output for seed 0, the published test vector 0xE220A8397B1DCDAF; (b) every round is one
    SplitMix64 step from state h + G*v, so the whole hash is a chain of `inputs.SplitMix64` (the generator that
    test_generator_check_values pins to the values SURVEY App. C prints)."""
    g = I.SplitMix64(0)
    assert g.next() == 0xE220A8397B1DCDAF and g.next() == 0x6E789E6AA1B965F4

    def chain(seed, vals):
        h = seed
        for v in vals:
            h = I.SplitMix64((h + I.GOLDEN * v) & I.MASK64).next()
        return (h >> 11) * 2.0 ** -53

    for seed, vals in ((0, (0, 0, 0, 0)), (1007, (0, 2, 5, 17)), (5007, (255, 8, 449, 0)), (2 ** 63 + 11, (3, 6, 14999, 1))):
        u = O.uniform(seed, *vals)
        assert 0.0 <= u < 1.0 and u == chain(seed, vals)
    # four rounds from seed 0 with v = 0: 0xE220A8397B1DCDAF -> ... -> 0x2130748aaac80268 (computed with Python integers)
    assert O.uniform(0, 0, 0, 0, 0) == (0x2130748aaac80268 >> 11) * 2.0 ** -53


def test_per_position_codon_weights():
    """orc_tt_build_pos (penalty on codon c 'at amino acid position i'): a per-residue table that repeats one
    row equals the shared table; adding delta to every codon of ONE residue shifts log Z by exactly delta (every sequence uses
    exactly one codon there); the weight sum equals direct enumeration."""
    m = I.tm1_model()
    aa = "RSLGS"
    cw = I.tm1_codon_logw()
    for kind, pw in ((0, None), (1, I.tm1_pair_logw())):
        base = O.inside(m, O.TT.build(aa, kind, cw, pw)).logZ
        tiled = np.tile(cw, (len(aa), 1))
        assert abs(O.inside(m, O.TT.build(aa, kind, tiled, pw)).logZ - base) < 1e-13
        shifted = tiled.copy()
        shifted[4] += 0.37  # the second S only
        assert abs(O.inside(m, O.TT.build(aa, kind, shifted, pw)).logZ - base - 0.37) < 1e-12
    # distinct rows: sum_phi W(phi) by direct enumeration over codon choices
    import itertools

    code = "KNKNTTTTRSRSIIMIQHQHPPPPRRRRLLLLEDEDAAAAGGGGVVVV*Y*YSSSS*CWCLFLF"
    rng = np.random.default_rng(7)
    cwp = rng.normal(0, 0.5, (4, 64))
    cods = [[c for c in range(64) if code[c] == a] for a in "RSLG"]
    tot = sum(math.exp(sum(cwp[k, c] for k, c in enumerate(ch))) for ch in itertools.product(*cods))
    assert abs(O.TT.build("RSLG", 0, cwp).logsum() - math.log(tot)) < 1e-12
    assert abs(O.TT.build("RSLG", 1, cwp).logsum() - math.log(tot)) < 1e-12


# ---------------------------------------------------------------- frequency matching (Alg S4.6)
def test_frequency_matching_fixed_point_vs_brute_force():
    """O.match_frequencies (PAPER.md Alg S4.6) against what the algorithm is for: with the returned bonuses the accumulated codon
    frequencies -- computed by explicit enumeration of every (sequence, structure), not by the routine's own marginals -- equal the
    targets; the first iterate is off by far more than the tolerance (the pairing model does bias codon usage), and the error
    of the naive iteration decreases."""
    m = I.tm1_model()
    rng = np.random.default_rng(3)
    logf_star = rng.normal(0.0, 0.7, 64)
    for aa, kind in (("RSLG", 0), ("LSR", 1)):
        pw = I.tm1_pair_logw() if kind else None
        logf, errs = O.match_frequencies(m, aa, kind, logf_star, pw, rtol=1e-8, max_iter=200)
        assert errs[0] > 1e-3 and errs[-1] < 1e-8 and (np.diff(errs[3:]) < 0).all()  # (the first steps may overshoot)
        bstar = O.target_frequencies(aa, logf_star)
        bf = O.brute_force(m, O.TT.build(aa, kind, logf, pw), marginals=True)
        np.testing.assert_allclose(bf["codon"].sum(0), bstar, atol=1e-7)
        assert abs(bstar.sum() - len(aa)) < 1e-12


# ---------------------------------------------------------------- minimisation (tropical semiring, eq 2.8)
@pytest.mark.parametrize("aa,kind,cw,pw", [("MW", 0, 0, 0), ("LSR", 0, 1, 0), ("LSR", 1, 1, 1), ("RSLG", 0, 1, 0), ("GRL", 1, 1, 1),
                                            ("MWFMWM", 0, 1, 0)])
def test_mfe_equals_enumeration(aa, kind, cw, pw):
    """orc_mfe (the recursion with (+, x) -> (min, +), PAPER.md S4d) against the definition: the smallest
    f = E/kT - log W over every (operator path, structure) by explicit enumeration; the returned state attains it
    (its own log-weight, evaluated by orc_logweight, equals -f_min); f_min >= -log Z."""
    m = I.tm1_model()
    m.ml_a = 0.4  # make multiloops competitive on these tiny designs
    tt = build(aa, kind, cw, pw)
    fb, sb, pb = O.mfe(m, tt, brute=True)
    fd, sd, pd = O.mfe(m, tt)
    assert abs(fd - fb) < 1e-12 * max(1.0, abs(fb))
    assert abs(-O.logweight(m, tt, sd, pd) - fd) < 1e-12 * max(1.0, abs(fd))
    assert abs(-O.logweight(m, tt, sb, pb) - fb) < 1e-12 * max(1.0, abs(fb))
    assert fd >= -O.inside(m, tt).logZ - 1e-12


def test_mfe_fixed_sequence_and_larger():
    """Beyond enumeration: for a Met/Trp protein (one sequence) the minimiser's energy is that sequence's structure MFE and no
    sampled structure of the same sequence lies below it; for a 13-aa design no sampled state lies below f_min."""
    m = I.nn_model()
    for aa, kind in (("MWMWMWMMWWMW", 0), (I.protein(1000, 13), 0), (I.protein(5000, 9), 1)):
        d = I.design(1 if kind == 0 else 5, 0, len(aa))
        tt = O.TT.build(aa, kind, d.codon_logw, d.pair_logw)
        f, s, p = O.mfe(m, tt)
        assert abs(-O.logweight(m, tt, s, p) - f) < 1e-11 * max(1.0, abs(f))
        tab = O.inside(m, tt)
        assert f >= -tab.logZ
        seqs, pairs = tab.sample(200, 77)
        lw = np.array([O.logweight(m, tt, seqs[k], pairs[k]) for k in range(200)])
        assert (-lw >= f - 1e-10).all()
