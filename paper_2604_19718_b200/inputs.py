"""Seeded synthetic input generators.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2604_19718_b200/csrc``).  It holds none of the method's arithmetic:
it only draws amino-acid strings, soft-constraint log-weights and nearest-
neighbour energy parameters from SplitMix64 streams, so that every test and the
bench see identical inputs on both sides.

The inputs stand in for the paper's random-protein benchmark (Fig 7
PAPER.md:270) and its CAI / CPB weight tables, none of which is in
the container; shapes follow BASELINE.json ``configs``.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

MASK64 = (1 << 64) - 1
GOLDEN = 0x9E3779B97F4A7C15
STREAM_MUL = 0xD1B54A32D192ED03
AMINO = "ACDEFGHIKLMNPQRSTVWY"

TAG_PROTEIN, TAG_CODON_W, TAG_PAIR_W, TAG_MODEL = 1, 2, 3, 4

TT_SINGLE_CODON = 0
TT_CODON_PAIR = 1

GAS_R = 8.31446261815324 / 4184.0  # kcal / (mol K)
T37 = 310.15


class SplitMix64:
    def __init__(self, seed: int, tag: int = 0):
        self.state = (seed ^ ((tag * STREAM_MUL) & MASK64)) & MASK64

    def next(self) -> int:
        self.state = (self.state + GOLDEN) & MASK64
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return (self.next() >> 11) * (2.0 ** -53)

    def normal(self) -> float:
        u1 = self.uniform()
        u2 = self.uniform()
        return math.sqrt(-2.0 * math.log(1.0 - u1)) * math.cos(2.0 * math.pi * u2)


def protein(seed: int, L: int) -> str:
    g = SplitMix64(seed, TAG_PROTEIN)
    return "".join(AMINO[int(20.0 * g.uniform())] for _ in range(L))


def codon_logw(seed: int, sigma: float = 0.5) -> np.ndarray:
    g = SplitMix64(seed, TAG_CODON_W)
    return np.array([sigma * g.normal() for _ in range(64)], dtype=np.float64)


def pair_logw(seed: int, sigma: float = 0.3) -> np.ndarray:
    g = SplitMix64(seed, TAG_PAIR_W)
    return np.array([sigma * g.normal() for _ in range(64 * 64)], dtype=np.float64).reshape(64, 64)


REV_PAIR = (3, 2, 1, 0, 5, 4)  # AU<->UA, CG<->GC, GU<->UG


@dataclass
class NNModel:
    """Plain container of nearest-neighbour parameters (kcal/mol)."""

    temperature_K: float = T37
    stack: np.ndarray = field(default_factory=lambda: np.zeros((6, 6)))
    tmm: np.ndarray = field(default_factory=lambda: np.zeros((6, 4, 4)))
    hairpin_a: float = 5.4
    hairpin_b: float = 1.75
    hairpin_l0: float = 9.0
    bulge_init: np.ndarray = field(default_factory=lambda: np.zeros(31))
    interior_init: np.ndarray = field(default_factory=lambda: np.zeros(31))
    ml_a: float = 3.4
    ml_b: float = 0.0
    ml_c: float = 0.4
    max_interior: int = 30
    min_hairpin: int = 3
    allow_all_pairs: int = 0

    @property
    def kT(self) -> float:
        return GAS_R * self.temperature_K


def _loop_inits(kT: float):
    bulge = np.zeros(31)
    interior = np.zeros(31)
    for l in range(1, 31):
        bulge[l] = 3.8 + 1.75 * kT * math.log(l)
    for l in range(2, 31):
        interior[l] = 2.0 + 1.75 * kT * math.log(l / 2.0)
    return bulge, interior


def nn_model(seed: int = 19718) -> NNModel:
    """Synthetic NN model of BASELINE.json configs[0]."""
    g = SplitMix64(seed, TAG_MODEL)
    m = NNModel()
    stack = np.zeros((6, 6))
    for p in range(6):
        for q in range(6):
            pp, qq = REV_PAIR[q], REV_PAIR[p]
            if (pp, qq) < (p, q):
                stack[p, q] = stack[pp, qq]
            else:
                stack[p, q] = -3.5 + 3.0 * g.uniform()
    tmm = np.zeros((6, 4, 4))
    for p in range(6):
        for x in range(4):
            for y in range(4):
                tmm[p, x, y] = -1.5 + 1.5 * g.uniform()
    m.stack, m.tmm = stack, tmm
    m.bulge_init, m.interior_init = _loop_inits(m.kT)
    return m


def tm1_model() -> NNModel:
    """Deterministic test model "TM1"."""
    m = NNModel()

    def s0(p, q):
        return 0.5 + 0.3 * p + 0.11 * q

    for p in range(6):
        for q in range(6):
            m.stack[p, q] = -0.5 - 0.5 * (s0(p, q) + s0(REV_PAIR[q], REV_PAIR[p]))
        for x in range(4):
            for y in range(4):
                m.tmm[p, x, y] = -0.1 * ((p + 2 * x + 3 * y) % 7)
    m.bulge_init, m.interior_init = _loop_inits(m.kT)
    return m


def tm1_codon_logw() -> np.ndarray:
    return np.array([0.1 * (i % 5) - 0.2 for i in range(64)], dtype=np.float64)


def tm1_pair_logw() -> np.ndarray:
    w = np.zeros((64, 64))
    for i in range(64):
        for j in range(64):
            w[i, j] = 0.05 * ((i + 2 * j) % 7) - 0.15
    return w


def zero_energy_model(allow_all_pairs: int = 1, max_interior: int = 30) -> NNModel:
    """All loop energies zero: Z = #sequences x #structures (closed-form pin)."""
    m = NNModel(hairpin_a=0.0, hairpin_b=0.0, ml_a=0.0, ml_b=0.0, ml_c=0.0)
    m.allow_all_pairs = allow_all_pairs
    m.max_interior = max_interior
    return m


@dataclass
class Design:
    """One design problem of BASELINE.json ``configs``."""

    name: str
    aa: str
    kind: int
    codon_logw: np.ndarray | None
    pair_logw: np.ndarray | None
    seed: int
    n_samples: int = 0

    @property
    def n(self) -> int:
        return 3 * len(self.aa)

    @property
    def sample_seed(self) -> int:
        return self.seed + 7


def design(config: int, item: int = 0, L: int | None = None) -> Design:
    """Design ``item`` of BASELINE.json configs[config-1] (1-based ``config``).

    ``L`` overrides the protein length (prefix-stable stream), used for the
    reduced-size parity cases.
    """
    seed = 1000 * config + item
    lengths = {1: 20, 2: 300, 3: 1000, 4: 5000, 5: 150}
    kinds = {1: TT_SINGLE_CODON, 2: TT_CODON_PAIR, 3: TT_CODON_PAIR, 4: TT_SINGLE_CODON, 5: TT_CODON_PAIR}
    samples = {1: 1000, 2: 0, 3: 0, 4: 100, 5: 256}
    LL = lengths[config] if L is None else L
    kind = kinds[config]
    return Design(
        name=f"config{config}_item{item}_L{LL}",
        aa=protein(seed, LL),
        kind=kind,
        codon_logw=codon_logw(seed),
        pair_logw=pair_logw(seed) if kind == TT_CODON_PAIR else None,
        seed=seed,
        n_samples=samples[config],
    )


def closed_form_inputs(kind: str, n: int):
    """Seeded inputs of the two large closed-form pins (tests/golden/make_golden.py closed, tests/test_gpu_parity.py):
    'zero8'  : generic operator list of bond dimension 8 (16 boundary states per position), n nucleotides; with the zero-energy,
               all-pairs model  Z = (sum_phi W(phi)) x S_30(n)  (BASELINE.json north_star "zero-energy closed forms");
    'mettrp' : protein of n/3 residues drawn from {M, W} (one codon each: a fixed sequence), codon weights of seed 424242; with the NN
               model  log Z = log Z_McCaskill(sequence) + sum of the codon log-weights (north_star "Met/Trp only")."""
    if kind == "zero8":
        ops = []
        for i in range(n):
            sa = 1 if i == 0 else 8
            sc = 1 if i == n - 1 else 8
            pos = []
            for a in range(sa):
                for b in (i % 4, (i + 1) % 4):
                    pos.append((a, b, (a + 3 * b + i) % sc, 0.5 + 0.03 * ((3 * a + 5 * b + i) % 11)))
            ops.append(pos)
        return ops
    g = SplitMix64(424242, TAG_PROTEIN)
    aa = "".join("MW"[g.next() & 1] for _ in range(n // 3))
    return aa, codon_logw(424242)


TAG_TENSOR_MODEL = 5


@dataclass
class TensorModel:
    """Parameters of the paper's tensor-based free-energy model (PAPER.md S2b lines 430-437; chi of eq 3.6): V[x] for an
    unpaired base x, B[x][y][rho] for the 5' side of a pair with 5' base x and 3' base y (B[y][x][rho] is its 3' side), S of the
    weighted trace Tr_S[X] = Tr[S X], gamma = model dimension, xi = number of pair conformations."""

    gamma: int
    xi: int
    V: np.ndarray          # [4][gamma][gamma]
    B: np.ndarray          # [4][4][xi][gamma][gamma], zero where x.y cannot pair
    S: np.ndarray          # [gamma][gamma]
    min_hairpin: int = 3   # B_{i,j} = 0 for |j - i| < 4


def tensor_model(gamma: int, xi: int, seed: int = 19718, unit: bool = False) -> TensorModel:
    """Synthetic non-negative parameters (the fitted parameters of ref [15] are not in the container): entries ~ U(0,1) scaled so
    that an unpaired step has row sums near 1 (the renormalisation of S3a, line 499, in spirit) and a canonical pair carries a
    weight of order e^{1..2}; ``unit`` = all-ones model of dimension 1 in which every two bases may pair (Z = number of sequences x number of structures)."""
    can = {(0, 3), (3, 0), (1, 2), (2, 1), (2, 3), (3, 2)}  # AU UA CG GC GU UG
    V = np.zeros((4, gamma, gamma))
    B = np.zeros((4, 4, xi, gamma, gamma))
    S = np.zeros((gamma, gamma))
    if unit:
        assert gamma == 1 and xi == 1
        V[:] = 1.0
        S[:] = 1.0
        B[:] = 1.0  # every two bases may pair: the structure counts S(n) of tests/golden/structure_counts.txt apply
        return TensorModel(gamma, xi, V, B, S)
    g = SplitMix64(seed, TAG_TENSOR_MODEL)
    for x in range(4):
        for a in range(gamma):
            for b in range(gamma):
                V[x, a, b] = (0.2 + g.uniform()) / (0.7 * gamma)
    strength = {(1, 2): 2.2, (2, 1): 2.2, (0, 3): 1.5, (3, 0): 1.5, (2, 3): 1.0, (3, 2): 1.0}
    for x in range(4):
        for y in range(4):
            for r in range(xi):
                for a in range(gamma):
                    for b in range(gamma):
                        u = g.uniform()
                        if (x, y) in can:
                            B[x, y, r, a, b] = strength[(x, y)] * (0.2 + u) / gamma
    for a in range(gamma):
        for b in range(gamma):
            S[a, b] = (1.0 if a == b else 0.0) + 0.15 * g.uniform()
    return TensorModel(gamma, xi, V, B, S)
