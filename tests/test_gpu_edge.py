"""GPU edge cases and statistical checks of the CUDA path (through the C ABI)."""
import math
from collections import Counter

import numpy as np
import pytest

from paper_2604_19718_b200 import inputs as I

pytestmark = pytest.mark.gpu
LOGZ_RTOL = 1e-9


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding, build

    build.build()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle

    return oracle


def _chi2_pvalue(stat, dof):
    from scipy.stats import chi2

    return float(chi2.sf(stat, dof))


@pytest.mark.parametrize("aa", ["M", "W", "L", "MW", "LL", "RS", "MWM"])
@pytest.mark.parametrize("kind", [0, 1])
def test_degenerate_lengths(B, O, aa, kind):
    """n = 3, 6, 9: no cell can close (hairpin >= 3 needs d >= 4 and a pairable combination): log Z = log sum_phi W(phi) or a few hairpins."""
    m = I.nn_model()
    cw, pw = I.codon_logw(7), (I.pair_logw(7) if kind else None)
    lo = O.inside(m, O.TT.build(aa, kind, cw, pw)).logZ
    tg, lz = B.inside(B.Model(m), B.TensorTrain.build(aa, kind, cw, pw))
    assert abs(lz - lo) <= LOGZ_RTOL * max(abs(lo), 1e-3)
    if len(aa) == 1:
        assert abs(lz - O.TT.build(aa, kind, cw, pw).logsum()) < 1e-12  # eq 3.2: no structure but the empty one
    s, p = tg.sample(16, 3)
    assert (s.cpu().numpy() < 4).all()


@pytest.mark.parametrize("aa", ["MWMWMWMWMWMW", "WWWWWWWWMMMMMMMM"])
def test_fixed_sequence_reduces_to_mccaskill(B, O, aa):
    """Single-codon protein (Met / Trp only): the design space has one sequence, Z = W x scalar McCaskill (north_star invariant)."""
    m = I.nn_model()
    cw = I.codon_logw(11)
    tt = O.TT.build(aa, 0, cw)
    seq = np.array(["ACGU".index(ch) for a in aa for ch in {"M": "AUG", "W": "UGG"}[a]], dtype=np.uint8)
    want = O.mccaskill(m, seq) + tt.logsum()
    for kind in (0, 1):
        tg, lz = B.inside(B.Model(m), B.TensorTrain.build(aa, kind, cw))
        assert abs(lz - want) <= LOGZ_RTOL * abs(want)
        s, p = tg.sample(8, 5)
        assert (s.cpu().numpy() == seq[None, :]).all()


def test_all_leucine_maximal_degeneracy(B, O):
    """Six-fold degenerate residues only: bond dimensions 2 / 4 (single) and 6 (pair) everywhere."""
    m = I.nn_model()
    aa = "L" * 14
    for kind in (0, 1):
        cw, pw = I.codon_logw(3), (I.pair_logw(3) if kind else None)
        lo = O.inside(m, O.TT.build(aa, kind, cw, pw)).logZ
        tg, lz = B.inside(B.Model(m), B.TensorTrain.build(aa, kind, cw, pw))
        assert abs(lz - lo) <= LOGZ_RTOL * abs(lo)


def test_generic_operators_bond_dimension_8(B, O):
    """cdz_tt_from_operators at the kernel limits: bond dimension 8, 16 boundary states per position."""
    m = I.tm1_model()
    n = 26
    ops = []
    for i in range(n):
        sa = 1 if i == 0 else 8
        sc = 1 if i == n - 1 else 8
        pos = []
        for a in range(sa):
            for b in (i % 4, (i + 1) % 4):  # two nucleotides per position: 8 x 2 left states, 2 x 8 right states
                c = (a + 3 * b + i) % sc
                pos.append((a, b, c, 0.5 + 0.03 * ((3 * a + 5 * b + i) % 11)))
        ops.append(pos)
    lo = O.inside(m, O.TT.from_ops(ops)).logZ
    tg, lz = B.inside(B.Model(m), B.TensorTrain.from_operators(ops))
    assert abs(lz - lo) <= LOGZ_RTOL * abs(lo)
    to = O.inside(m, O.TT.from_ops(ops))
    so, po = to.sample(64, 9)
    sg, pg = tg.sample(64, 9)
    assert (sg.cpu().numpy() == so).all() and (pg.cpu().numpy() == po).all()


def test_invalid_inputs_are_rejected(B):
    with pytest.raises(B.CdzError):
        B.TensorTrain.build("MXW", 0)  # unknown residue
    with pytest.raises(B.CdzError):
        B.TensorTrain.build("MW", 0, np.full(64, np.nan))
    with pytest.raises(B.CdzError):
        B.TensorTrain.from_operators([[(0, 0, 0, 1.0)], [(0, 5, 0, 1.0)]])  # nucleotide out of range
    bad = I.nn_model()
    bad.max_interior = 31
    with pytest.raises(B.CdzError):
        B.Model(bad)
    tt = B.TensorTrain.build("MW", 0)
    with pytest.raises(B.CdzError):
        B.inside(B.Model(I.nn_model()), tt, precision=7)  # unknown precision code


@pytest.mark.parametrize("aa,kind", [("RSLG", 0), ("LSR", 1)])
def test_gpu_samples_follow_the_exact_joint_distribution(B, O, aa, kind):
    """chi-square of 40000 GPU samples against p = W e^{-E/kT} / Z evaluated state by state with the oracle's energy function."""
    m = I.tm1_model()
    m.ml_a = 0.4
    cw, pw = I.tm1_codon_logw(), (I.tm1_pair_logw() if kind else None)
    tto = O.TT.build(aa, kind, cw, pw)
    tg, lz = B.inside(B.Model(m), B.TensorTrain.build(aa, kind, cw, pw))
    J = 40000
    seq, pair = tg.sample(J, 4242)
    seq, pair = seq.cpu().numpy(), pair.cpu().numpy()
    cnt = Counter((s.tobytes(), p.tobytes()) for s, p in zip(seq, pair))
    stat, dof, seen_p, pool_e, pool_o = 0.0, 0, 0.0, 0.0, 0.0
    for (sb, pb), c in cnt.items():
        lw = O.logweight(m, tto, np.frombuffer(sb, dtype=np.uint8), np.frombuffer(pb, dtype=np.int32))
        assert np.isfinite(lw), "sampled an invalid state"
        pr = math.exp(lw - lz)
        seen_p += pr
        e = J * pr
        if e >= 10:
            stat += (c - e) ** 2 / e
            dof += 1
        else:
            pool_e += e
            pool_o += c
    pool_e += J * max(0.0, 1.0 - seen_p)
    if pool_e >= 10:
        stat += (pool_o - pool_e) ** 2 / pool_e
        dof += 1
    assert dof > 5 and _chi2_pvalue(stat, dof - 1) > 1e-3


def test_gpu_sample_marginals_vs_brute_force(B, O):
    """Codon and unpaired frequencies of GPU samples vs the exact brute-force marginals (4-aa prefix of config 1); zero mass on
    disallowed codons."""
    m = I.nn_model()
    d = I.design(1, 0, 4)
    bf = O.brute_force(m, O.TT.build(d.aa, d.kind, d.codon_logw), marginals=True)
    tg, lz = B.inside(B.Model(m), B.TensorTrain.build(d.aa, d.kind, d.codon_logw))
    assert abs(lz - bf["logZ"]) <= LOGZ_RTOL * abs(bf["logZ"])
    J = 20000
    seq, pair = tg.sample(J, d.sample_seed)
    seq, pair = seq.cpu().numpy(), pair.cpu().numpy()
    stat, dof = 0.0, 0
    for k in range(len(d.aa)):
        cod = 16 * seq[:, 3 * k].astype(int) + 4 * seq[:, 3 * k + 1] + seq[:, 3 * k + 2]
        obs = np.bincount(cod, minlength=64)
        assert obs[bf["codon"][k] == 0].sum() == 0
        e = J * bf["codon"][k]
        big = e >= 5
        if big.sum() >= 2:
            stat += ((obs[big] - e[big]) ** 2 / e[big]).sum()
            dof += big.sum() - 1
    np.testing.assert_allclose((pair < 0).mean(0), np.diag(bf["bpp"]), atol=5 * 0.5 / math.sqrt(J))
    assert _chi2_pvalue(stat, dof) > 1e-3
