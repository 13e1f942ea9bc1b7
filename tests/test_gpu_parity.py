"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element."""
import math
import os

import numpy as np
import pytest

from paper_2604_19718_b200 import inputs as I

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden")
LOGZ_RTOL = 1e-9  # BASELINE.json north_star: 1e-9 relative in log Z for fp64


def rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


@pytest.fixture(scope="module")
def B():
    from paper_2604_19718_b200 import binding, build

    build.build()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle

    return oracle


_ORACLE_TABLES = {}


def oracle_design(O, cfg, L):
    """Oracle inside pass of a BASELINE design prefix under the NN model; computed once per process for the sizes several tests share
    (the long-double recursion dominates the run time of this file)."""
    key = (cfg, L)
    if key in _ORACLE_TABLES:
        return _ORACLE_TABLES[key]
    d = I.design(cfg, 0, L)
    to = O.inside(I.nn_model(), O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    if d.n <= 300:
        _ORACLE_TABLES[key] = to
    return to


def both_design(B, O, cfg, L):
    d = I.design(cfg, 0, L)
    tg, lz = B.inside(B.Model(I.nn_model()), B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    return oracle_design(O, cfg, L), tg, lz


def both(B, O, model, aa, kind, cw, pw):
    tto = O.TT.build(aa, kind, cw, pw)
    ttg = B.TensorTrain.build(aa, kind, cw, pw)
    to = O.inside(model, tto)
    tg, lz = B.inside(B.Model(model), ttg)
    return to, tg, lz


@pytest.mark.parametrize("row", rows("appendix_b.txt"), ids=lambda r: "-".join(r[:5]))
def test_logz_appendix_b(B, O, row):
    aa, kind, cw, pw, mi = row[0], int(row[1]), int(row[2]), int(row[3]), int(row[4])
    m = I.tm1_model()
    m.max_interior = mi
    to, tg, lz = both(B, O, m, aa, kind, I.tm1_codon_logw() if cw else None, I.tm1_pair_logw() if pw else None)
    assert abs(lz - to.logZ) <= LOGZ_RTOL * max(abs(to.logZ), 1e-3)
    assert abs(lz - float(row[5])) <= 1e-9 * max(1.0, abs(float(row[5])))


@pytest.mark.parametrize("cfg,L", [(1, 20), (2, 20), (5, 10), (5, 40), (2, 45), (1, 67), (1, 150), (2, 100)])
def test_logz_and_tables_vs_oracle(B, O, cfg, L):
    """Every stored cell (Qb, Qbs, Qm1, Qml, M2, Qm) of every (i,j) agrees with the oracle."""
    d = I.design(cfg, 0, L)
    to, tg, lz = both_design(B, O, cfg, L)
    assert abs(lz - to.logZ) <= LOGZ_RTOL * abs(to.logZ)
    n = d.n
    rng = np.random.default_rng(0)
    cells = [(i, j) for i in range(n) for j in range(i, n)]
    if len(cells) > 1500:
        idx = rng.choice(len(cells), 1500, replace=False)
        cells = [cells[k] for k in idx] + [(0, n - 1), (1, n - 2), (0, n - 2)]
    for (i, j) in cells:
        for which in range(6):
            g, sh = tg.cell(which, i, j)
            o = to.cell(which, i, j, sh)
            scale = max(np.abs(o).max(), 1e-300)
            assert np.abs(g - o).max() <= 1e-11 * scale, (which, i, j)
    for j in (0, n // 2, n - 1):
        for c in range(1):
            assert abs(tg.logqext(j, c) - to.logqext(j, c)) <= 1e-11 * max(1.0, abs(to.logqext(j, c)))


@pytest.mark.parametrize("n", [12, 24, 37, 40, 50])
def test_zero_energy_closed_form(B, O, n):
    """Z = #structures for one fixed sequence, all pairs allowed, zero energies (tests/golden/structure_counts.txt)."""
    tab = {(k, int(a)): int(v) for k, a, v in rows("structure_counts.txt")}
    m = I.zero_energy_model()
    tt = B.TensorTrain.from_operators([[(0, 0, 0, 1.0)]] * n)
    tg, lz = B.inside(B.Model(m), tt)
    want = tab[("limit30", n)] if n >= 38 else tab[("unlimited", n)]
    assert abs(math.exp(lz) / want - 1) < 1e-12


def test_zero_energy_sequences_times_structures(B, O):
    m = I.zero_energy_model()
    for aa, want in (("LSR", 6912), ("RSLG", 236736), ("GAVLI", 2858112)):
        for kind in (0, 1):
            tg, lz = B.inside(B.Model(m), B.TensorTrain.build(aa, kind))
            assert abs(math.exp(lz) / want - 1) < 1e-12


def test_generic_operator_lists(B, O):
    m = I.tm1_model()
    ops = [[(0, b, 0, 1.0 + 0.1 * b + 0.01 * i) for b in range(4)] for i in range(14)]
    lo = O.inside(m, O.TT.from_ops(ops)).logZ
    tg, lz = B.inside(B.Model(m), B.TensorTrain.from_operators(ops))
    assert abs(lz - lo) <= LOGZ_RTOL * abs(lo)


@pytest.mark.parametrize("cfg,L,J", [(1, 20, 1000), (5, 12, 300), (2, 20, 300), (5, 40, 64)])
def test_samples_bit_exact(B, O, cfg, L, J):
    """Same seed, same decision uniforms -> identical (sequence, structure) as the oracle traceback."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    to, tg, lz = both_design(B, O, cfg, L)
    so, po = to.sample(J, d.sample_seed)
    sg, pg = tg.sample(J, d.sample_seed)
    sg, pg = sg.cpu().numpy(), pg.cpu().numpy()
    bad = [k for k in range(J) if not ((so[k] == sg[k]).all() and (po[k] == pg[k]).all())]
    assert not bad, f"{len(bad)} of {J} samples differ, first {bad[:3]}"
    # every sample is a valid state of the ensemble
    tto = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    for k in range(0, J, max(1, J // 20)):
        assert np.isfinite(O.logweight(m, tto, sg[k], pg[k]))
    # determinism
    sg2, pg2 = tg.sample(J, d.sample_seed)
    assert (sg2.cpu().numpy() == sg).all() and (pg2.cpu().numpy() == pg).all()


def test_errors(B):
    m = B.Model(I.nn_model())
    tt = B.TensorTrain.build("MW", 0)
    tg, lz = B.inside(m, tt)
    with pytest.raises(B.CdzError):
        tg.cell(9, 0, 0)


# ---- BASELINE.json full sizes: what the oracle can still reach, plus properties that hold at any size -------------------
def _prefix_chain(B, O, cfg, L_full, L_pre, rtol=1e-11):
    """log Qext(j)[c] depends on positions <= j only, so the full-size GPU run restricted to a prefix must equal an
    independent GPU run on that prefix, which in turn is checked element-wise against the oracle (last row)."""
    m = I.nn_model()
    d = I.design(cfg, 0, L_full)
    dp = I.design(cfg, 0, L_pre)
    assert d.aa.startswith(dp.aa)
    tfull, lz_full = B.inside(B.Model(m), B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    to, tpre, lz_pre = both(B, O, m, dp.aa, dp.kind, dp.codon_logw, dp.pair_logw)
    assert abs(lz_pre - to.logZ) <= LOGZ_RTOL * abs(to.logZ)
    sig, _, _ = B.TensorTrain.build(dp.aa, dp.kind, dp.codon_logw, dp.pair_logw).describe()
    for j in sorted({0, dp.n // 3, dp.n // 2, dp.n - 2}):  # (the last bond of the prefix run is summed differently)
        for c in range(sig[j + 1]):
            ref = to.logqext(j, c)
            assert abs(tpre.logqext(j, c) - ref) <= rtol * max(1.0, abs(ref))
            assert abs(tfull.logqext(j, c) - ref) <= 1e-9 * max(1.0, abs(ref)), (j, c)
    return tfull, lz_full, d


def test_config4_full_size_prefix_and_samples(B, O):
    """configs[3]: 5000 aa (15000 nt), the launch configuration bench.py times: prefix chain to the oracle, every one
    of the 100 samples is a valid state with a finite Boltzmann weight, the pass is deterministic."""
    tfull, lz, d = _prefix_chain(B, O, 4, 5000, 60)
    assert np.isfinite(lz) and 1.2 * d.n < lz < 1.5 * d.n  # ~1.33 nat / nt with this model (SURVEY c-12)
    info = tfull.info()
    assert info["n"] == 15000 and info["n_rescales"] >= 8
    seq, pair = tfull.sample(100, d.sample_seed)
    seq, pair = seq.cpu().numpy(), pair.cpu().numpy()
    tto = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    m = I.nn_model()
    for k in range(100):  # every sample: a coding sequence of the protein with a valid structure of finite weight
        assert (seq[k] < 4).all()
        assert np.isfinite(O.logweight(m, tto, seq[k], pair[k]))
    tfull.rerun()
    assert tfull.logz() == lz


def test_config2_full_size_prefix(B, O):
    """configs[1]: 300 aa, codon-pair tensor train (bond dimension up to 6)."""
    _prefix_chain(B, O, 2, 300, 30)


def test_config3_size_runs_in_fp64(B, O):
    """configs[2] (1000 aa, codon-pair TT) is run through the fp64 path: prefix chain + finite log Z."""
    tfull, lz, d = _prefix_chain(B, O, 3, 1000, 30)
    assert np.isfinite(lz)


def test_batch_equals_single_and_oracle(B, O):
    """configs[4]: independent designs advanced in the same launches give exactly the single-design results."""
    m = I.nn_model()
    mg = B.Model(m)
    ds = [I.design(5, item, 24) for item in range(6)]
    tts = [B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw) for d in ds]
    tabs, lzs = B.inside_batch(mg, tts)
    for d, tt, tab, lz in zip(ds, tts, tabs, lzs):
        t1, lz1 = B.inside(mg, tt)
        assert lz == lz1
        lo = O.inside(m, O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)).logZ
        assert abs(lz - lo) <= LOGZ_RTOL * abs(lo)
        s1, p1 = t1.sample(32, d.sample_seed)
        s2, p2 = tab.sample(32, d.sample_seed)
        assert (s1 == s2).all() and (p1 == p2).all()


def test_batch_many_blocks_split_k_scratch(B):
    """with B > 1 the wave-aware split-K choice can pick more splits than a single-design launch; the partial-tile
    scratch GP must hold them.  NB >= 48 blocks, B = 12: batched == single, bit for bit."""
    m = I.nn_model()
    mg = B.Model(m)
    ds = [I.design(2, item, 350) for item in range(12)]  # codon-pair TT, ~50 blocks
    tts = [B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw) for d in ds]
    tabs, lzs = B.inside_batch(mg, tts)
    assert tabs[0].info()["n"] == 1050
    for item in (0, 5, 11):
        t1, lz1 = B.inside(mg, tts[item])
        assert abs(lzs[item] - lz1) <= 1e-12 * abs(lz1)
        n = ds[item].n
        for (i, j) in ((0, n - 1), (10, n - 20), (n // 3, 2 * n // 3), (400, 900)):
            for which in (0, 4, 5):
                g, sh = tabs[item].cell(which, i, j)
                g1, sh1 = t1.cell(which, i, j)
                # (the number of K-splits differs between the two launches, so the sums associate differently: last bits may differ)
                assert sh == sh1 and np.abs(g - g1).max() <= 1e-12 * max(np.abs(g1).max(), 1e-300)


def test_batch_mixed_lengths(B, O):
    """designs of different length in one batch; a shorter design that has finished must not be rescaled again
    at the later events of the longer ones.  Lengths chosen so that powers of two fall between the block counts."""
    m = I.nn_model()
    mg = B.Model(m)
    ds = [I.design(5, 0, 24), I.design(5, 1, 100), I.design(2, 0, 300), I.design(5, 2, 60)]
    tts = [B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw) for d in ds]
    tabs, lzs = B.inside_batch(mg, tts)
    for d, tt, tab, lz in zip(ds, tts, tabs, lzs):
        t1, lz1 = B.inside(mg, tt)
        assert lz == lz1, (d.name, lz, lz1)
        s1, p1 = t1.sample(16, d.sample_seed)
        s2, p2 = tab.sample(16, d.sample_seed)
        assert (s1 == s2).all() and (p1 == p2).all()
    lo = O.inside(m, O.TT.build(ds[0].aa, ds[0].kind, ds[0].codon_logw, ds[0].pair_logw)).logZ
    assert abs(lzs[0] - lo) <= LOGZ_RTOL * abs(lo)


def test_config5_full_batch(B, O):
    """64 x 150 aa in one batched pass: equal to the designs run one at a time; item 0's prefix checked against the oracle."""
    m = I.nn_model()
    mg = B.Model(m)
    ds = [I.design(5, item) for item in range(64)]
    tts = [B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw) for d in ds]
    tabs, lzs = B.inside_batch(mg, tts)
    assert all(np.isfinite(v) for v in lzs)
    for item in (0, 17, 63):
        t1, lz1 = B.inside(mg, tts[item])
        assert lzs[item] == lz1
    _prefix_chain(B, O, 5, 150, 20)


def _stored_oracle_rows():
    path = os.path.join(GOLD, "oracle_logz.txt")
    return rows("oracle_logz.txt") if os.path.exists(path) else []


@pytest.mark.parametrize("row", _stored_oracle_rows(), ids=lambda r: f"config{r[0]}-L{r[2]}")
def test_full_size_logz_vs_stored_oracle(B, row):
    """log Z of whole BASELINE designs against the value the plain CPU oracle computed for them (minutes to hours of CPU time,
    hence stored: tests/golden/oracle_logz.txt, written by tests/golden/make_golden.py which calls only oracle/)."""
    cfg, item, L, want = int(row[0]), int(row[1]), int(row[2]), float(row[4])
    d = I.design(cfg, item, L)
    assert d.n == int(row[3])
    tg, lz = B.inside(B.Model(I.nn_model()), B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    assert abs(lz - want) <= LOGZ_RTOL * abs(want), (lz, want)


def _stored_sample_rows():
    path = os.path.join(GOLD, "oracle_samples.txt")
    return rows("oracle_samples.txt") if os.path.exists(path) else []


@pytest.mark.parametrize("row", _stored_sample_rows(), ids=lambda r: f"config{r[0]}-J{r[3]}")
def test_full_size_samples_vs_stored_oracle(B, row):
    """Bit-exact samples at the BASELINE sizes the oracle can reach (config 1: 1000 x 60 nt; config 5 item 0: 256 x 450 nt, 15 blocks,
    multiloop-segment skip and 32-wide prefix sums exercised): SHA-256 of the raw arrays orc_sample produced for the same seed
    (tests/golden/oracle_samples.txt, written by tests/golden/make_golden.py samples; oracle only), plus sample 0 as text."""
    import hashlib

    cfg, item, L, J, seed = (int(v) for v in row[:5])
    d = I.design(cfg, item, L)
    assert d.sample_seed == seed and d.n_samples == J
    tg, lz = B.inside(B.Model(I.nn_model()), B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    seq, pair = tg.sample(J, seed)
    seq, pair = seq.cpu().numpy(), pair.cpu().numpy()
    assert "".join("ACGU"[b] for b in seq[0]) == row[7]
    assert "".join("." if q < 0 else ("(" if q > k else ")") for k, q in enumerate(pair[0])) == row[8]
    assert hashlib.sha256(seq.astype("uint8").tobytes()).hexdigest() == row[5]
    assert hashlib.sha256(pair.astype("<i4").tobytes()).hexdigest() == row[6]


# ---- large pins that do not go through the tensor recursion of the oracle ---------------------------------------
def _closed_rows():
    path = os.path.join(GOLD, "oracle_closed_forms.txt")
    return rows("oracle_closed_forms.txt") if os.path.exists(path) else []


@pytest.mark.parametrize("row", _closed_rows(), ids=lambda r: f"{r[0]}-{r[1]}")
def test_closed_form_large(B, row):
    """zero8: zero-energy, all-pairs model on a generic bond-dimension-8 operator list (16 boundary states per position): every
    sequence has the same number of structures, so  log Z = log sum_phi W(phi) + log S_30(n)  (orc_tt_logsum, eq 3.2, + the scalar
    orc_mccaskill count).  At n = 3000 this is 375 blocks: every block diagonal, 16-way split-K and the rescale events up to D = 256
    of the headline run, against a closed form.   mettrp: Met/Trp-only protein (one codon each) under the NN model: the design space
    is one sequence, log Z = scalar McCaskill + codon log-weights (north_star).  Expected values: tests/golden/oracle_closed_forms.txt
    (make_golden.py closed; oracle only)."""
    closed_form_inputs = I.closed_form_inputs

    kind, n, want = row[0], int(row[1]), float(row[2])
    if kind == "zero8":
        m = I.zero_energy_model()
        tt = B.TensorTrain.from_operators(closed_form_inputs("zero8", n))
    else:
        m = I.nn_model()
        aa, cw = closed_form_inputs("mettrp", n)
        tt = B.TensorTrain.build(aa, B.TT_SINGLE_CODON, cw)
    tg, lz = B.inside(B.Model(m), tt)
    assert abs(lz - want) <= LOGZ_RTOL * abs(want), (lz, want)
    tg.destroy()


@pytest.mark.parametrize("row", _closed_rows(), ids=lambda r: f"{r[0]}-{r[1]}")
def test_closed_form_large_fp32_scaled(B, row):
    """The same closed forms through CDZ_FP32_SCALED (3xTF32 split-point contraction, BASELINE configs[2] tolerance 1e-4): at 3000 nt the
    fp32 path is pinned to a value that owes nothing to the fp64 GPU path (the plain oracle cannot reach the 3000-nt codon-pair design)."""
    kind, n, want = row[0], int(row[1]), float(row[2])
    if kind == "zero8":
        m = I.zero_energy_model()
        tt = B.TensorTrain.from_operators(I.closed_form_inputs("zero8", n))
    else:
        m = I.nn_model()
        aa, cw = I.closed_form_inputs("mettrp", n)
        tt = B.TensorTrain.build(aa, B.TT_SINGLE_CODON, cw)
    tg, lz = B.inside(B.Model(m), tt, precision=B.FP32_SCALED)
    assert tg.info()["precision"] == B.FP32_SCALED
    assert abs(lz - want) <= FP32_RTOL * abs(want), (lz, want)
    tg.destroy()


@pytest.mark.parametrize("cfg", [2, 4])
def test_rescale_schedule_invariance(B, cfg):
    """The per-position scales are exact powers of two, so moving the rescale events (after block diagonals 1,2,4,.. -> 3,6,12,.. ->
    5,10,20,..) must leave log Z unchanged to rounding: 1e-12 relative at config 2 (900 nt) and at the headline config 4 (15000 nt)."""
    d = I.design(cfg, 0)
    tg, lz = B.inside(B.Model(I.nn_model()), B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw))
    n0 = tg.info()["n_rescales"]
    for first in (3, 5):
        tg.set_rescale_start(first)
        tg.rerun()
        lz2 = tg.logz()
        assert abs(lz2 - lz) <= 1e-12 * abs(lz), (first, lz, lz2)
        assert tg.info()["n_rescales"] != n0 or cfg == 2
    tg.destroy()


# ---- CDZ_FP32_SCALED: single-precision split-point contraction (BASELINE.json configs[2], tolerance 1e-4 relative in log Z) ---------
FP32_RTOL = 1e-4


@pytest.mark.parametrize("cfg,L", [(1, 20), (5, 40), (2, 100), (1, 200), (5, 150), (2, 300)])
def test_fp32_scaled_vs_oracle_and_fp64(B, O, cfg, L):
    """The fp32-scaled path against the oracle where it finishes in seconds (or is stored) and against the fp64 GPU path."""
    m = I.nn_model()
    d = I.design(cfg, 0, L)
    tt = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    t32, lz32 = B.inside(B.Model(m), tt, precision=B.FP32_SCALED)
    t64, lz64 = B.inside(B.Model(m), tt)
    assert abs(lz32 - lz64) <= FP32_RTOL * abs(lz64)
    assert t32.info()["precision"] == B.FP32_SCALED
    if d.n <= 300:
        lo = oracle_design(O, cfg, L).logZ
        assert abs(lz32 - lo) <= FP32_RTOL * abs(lo)
    stored = {(int(r[0]), int(r[2])): float(r[4]) for r in _stored_oracle_rows()}
    if (cfg, L) in stored:
        assert abs(lz32 - stored[(cfg, L)]) <= FP32_RTOL * abs(stored[(cfg, L)])
    # samples drawn from the fp32-contracted tables are valid states
    if d.n <= 450:
        seq, pair = t32.sample(8, d.sample_seed)
        tto = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
        for k in range(8):
            assert np.isfinite(O.logweight(m, tto, seq[k].cpu().numpy(), pair[k].cpu().numpy()))


def test_fp32_scaled_config3_and_config4(B):
    """configs[2] (1000 aa, codon-pair TT, 3000 nt) through the fp32-scaled path: against the fp64 GPU path and, when the hours-long
    oracle run has been stored (tests/golden/oracle_logz.txt), against the oracle; the same at the headline size."""
    stored = {(int(r[0]), int(r[2])): float(r[4]) for r in _stored_oracle_rows()}
    for cfg in (3, 4):
        d = I.design(cfg, 0)
        tt = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
        t32, lz32 = B.inside(B.Model(I.nn_model()), tt, precision=B.FP32_SCALED)
        t32.destroy()
        t64, lz64 = B.inside(B.Model(I.nn_model()), tt)
        t64.destroy()
        assert abs(lz32 - lz64) <= FP32_RTOL * abs(lz64), (cfg, lz32, lz64)
        if (cfg, len(d.aa)) in stored:
            want = stored[(cfg, len(d.aa))]
            assert abs(lz32 - want) <= FP32_RTOL * abs(want)
            assert abs(lz64 - want) <= LOGZ_RTOL * abs(want)
        print(f"config {cfg}: fp32-scaled {lz32:.9f} fp64 {lz64:.9f} rel diff {abs(lz32 - lz64) / abs(lz64):.2e}")
