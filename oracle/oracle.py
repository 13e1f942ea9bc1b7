"""ctypes wrapper of the CPU oracle (test infrastructure, NOT the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never imports paper_2604_19718_b200's CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class OrcModel(C.Structure):
    _fields_ = [
        ("temperature_K", C.c_double),
        ("stack", C.c_double * 36),
        ("tmm", C.c_double * 96),
        ("hairpin_a", C.c_double),
        ("hairpin_b", C.c_double),
        ("hairpin_l0", C.c_double),
        ("bulge_init", C.c_double * 31),
        ("interior_init", C.c_double * 31),
        ("ml_a", C.c_double),
        ("ml_b", C.c_double),
        ("ml_c", C.c_double),
        ("max_interior", C.c_int),
        ("min_hairpin", C.c_int),
        ("allow_all_pairs", C.c_int),
    ]


class OrcOp(C.Structure):
    _fields_ = [("a", C.c_int), ("b", C.c_int), ("c", C.c_int), ("x", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.orc_tt_build.argtypes = [C.c_char_p, C.c_int, C.c_int, dp, dp, C.POINTER(vp)]
        L.orc_tt_build_pos.argtypes = [C.c_char_p, C.c_int, C.c_int, dp, dp, C.POINTER(vp)]
        L.orc_tt_from_ops.argtypes = [C.c_int, ip, C.POINTER(OrcOp), C.POINTER(vp)]
        L.orc_tt_free.argtypes = [vp]
        L.orc_tt_n.argtypes = [vp]
        L.orc_tt_nops.argtypes = [vp]
        L.orc_tt_get.argtypes = [vp, ip, ip, C.POINTER(OrcOp)]
        L.orc_tt_logsum.argtypes = [vp]
        L.orc_tt_logsum.restype = C.c_double
        u8p, i32p = C.POINTER(C.c_uint8), C.POINTER(C.c_int32)
        L.orc_energy.argtypes = [C.POINTER(OrcModel), C.c_int, u8p, i32p, ip]
        L.orc_energy.restype = C.c_double
        L.orc_logweight.argtypes = [C.POINTER(OrcModel), vp, u8p, i32p]
        L.orc_logweight.restype = C.c_double
        L.orc_brute_force.argtypes = [C.POINTER(OrcModel), vp, dp, dp, dp, dp, dp]
        L.orc_count_structures.argtypes = [C.c_int, C.c_int, C.c_int]
        L.orc_count_structures.restype = C.c_double
        L.orc_mccaskill.argtypes = [C.POINTER(OrcModel), C.c_int, u8p]
        L.orc_mccaskill.restype = C.c_double
        L.orc_inside.argtypes = [C.POINTER(OrcModel), vp, C.c_int, C.POINTER(vp), dp]
        L.orc_tables_free.argtypes = [vp]
        L.orc_tables_cell.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, dp]
        L.orc_tables_logqext.argtypes = [vp, C.c_int, C.c_int]
        L.orc_tables_logqext.restype = C.c_double
        L.orc_sample.argtypes = [vp, C.c_int, C.c_uint64, u8p, i32p]
        L.orc_uniform.argtypes = [C.c_uint64] * 5
        L.orc_uniform.restype = C.c_double
        L.orc_marginals.argtypes = [vp, dp, dp, dp]
        L.orc_mfe.argtypes = [C.POINTER(OrcModel), vp, C.c_int, dp, u8p, i32p]
        L.orc_brute_force_min.argtypes = [C.POINTER(OrcModel), vp, dp, u8p, i32p]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def make_model(m) -> OrcModel:
    """Marshal an inputs.NNModel-like object (attributes only) into the oracle's struct."""
    s = OrcModel()
    s.temperature_K = float(m.temperature_K)
    s.stack[:] = [float(v) for v in np.asarray(m.stack, dtype=np.float64).reshape(-1)]
    s.tmm[:] = [float(v) for v in np.asarray(m.tmm, dtype=np.float64).reshape(-1)]
    s.hairpin_a, s.hairpin_b, s.hairpin_l0 = float(m.hairpin_a), float(m.hairpin_b), float(m.hairpin_l0)
    s.bulge_init[:] = [float(v) for v in np.asarray(m.bulge_init, dtype=np.float64)]
    s.interior_init[:] = [float(v) for v in np.asarray(m.interior_init, dtype=np.float64)]
    s.ml_a, s.ml_b, s.ml_c = float(m.ml_a), float(m.ml_b), float(m.ml_c)
    s.max_interior, s.min_hairpin, s.allow_all_pairs = int(m.max_interior), int(m.min_hairpin), int(m.allow_all_pairs)
    return s


class TT:
    def __init__(self, handle):
        self.h = handle
        self.n = lib().orc_tt_n(handle)

    @classmethod
    def build(cls, aa: str, kind: int, codon_logw=None, pair_logw=None) -> "TT":
        h = C.c_void_p()
        cw = np.ascontiguousarray(codon_logw, dtype=np.float64) if codon_logw is not None else None
        pw = np.ascontiguousarray(pair_logw, dtype=np.float64).reshape(-1) if pair_logw is not None else None
        if cw is not None and cw.ndim == 2:
            assert cw.shape == (len(aa), 64)
            rc = lib().orc_tt_build_pos(aa.encode(), len(aa), kind, _dp(cw.reshape(-1)), _dp(pw), C.byref(h))
        else:
            rc = lib().orc_tt_build(aa.encode(), len(aa), kind, _dp(cw), _dp(pw), C.byref(h))
        if rc != 0:
            raise ValueError(f"orc_tt_build failed rc={rc}")
        return cls(h)

    @classmethod
    def from_ops(cls, ops_per_pos) -> "TT":
        n = len(ops_per_pos)
        counts = (C.c_int * n)(*[len(o) for o in ops_per_pos])
        flat = [o for pos in ops_per_pos for o in pos]
        arr = (OrcOp * max(1, len(flat)))()
        for k, (a, b, c, x) in enumerate(flat):
            arr[k] = OrcOp(a, b, c, x)
        h = C.c_void_p()
        rc = lib().orc_tt_from_ops(n, counts, arr, C.byref(h))
        if rc != 0:
            raise ValueError("orc_tt_from_ops failed")
        return cls(h)

    def get(self):
        n, nops = self.n, lib().orc_tt_nops(self.h)
        sigma = (C.c_int * (n + 1))()
        counts = (C.c_int * n)()
        ops = (OrcOp * max(1, nops))()
        lib().orc_tt_get(self.h, sigma, counts, ops)
        out, k = [], 0
        for i in range(n):
            out.append([(ops[k + t].a, ops[k + t].b, ops[k + t].c, ops[k + t].x) for t in range(counts[i])])
            k += counts[i]
        return list(sigma), out

    def logsum(self) -> float:
        return lib().orc_tt_logsum(self.h)

    def __del__(self):
        try:
            lib().orc_tt_free(self.h)
        except Exception:
            pass


def energy(model, seq, pair):
    seq = np.ascontiguousarray(seq, dtype=np.uint8)
    pair = np.ascontiguousarray(pair, dtype=np.int32)
    valid = C.c_int()
    m = make_model(model)
    e = lib().orc_energy(C.byref(m), len(seq), seq.ctypes.data_as(C.POINTER(C.c_uint8)),
                         pair.ctypes.data_as(C.POINTER(C.c_int32)), C.byref(valid))
    return e, bool(valid.value)


def logweight(model, tt: TT, seq, pair) -> float:
    seq = np.ascontiguousarray(seq, dtype=np.uint8)
    pair = np.ascontiguousarray(pair, dtype=np.int32)
    m = make_model(model)
    return lib().orc_logweight(C.byref(m), tt.h, seq.ctypes.data_as(C.POINTER(C.c_uint8)),
                               pair.ctypes.data_as(C.POINTER(C.c_int32)))


def brute_force(model, tt: TT, marginals: bool = False):
    n = tt.n
    m = make_model(model)
    logZ, ns = C.c_double(), C.c_double()
    bpp = np.zeros((n, n)) if marginals else None
    base = np.zeros((n, 4)) if marginals else None
    codon = np.zeros((n // 3, 64)) if marginals else None
    lib().orc_brute_force(C.byref(m), tt.h, C.byref(logZ), _dp(bpp), _dp(base), _dp(codon), C.byref(ns))
    return dict(logZ=logZ.value, n_states=ns.value, bpp=bpp, base=base, codon=codon)


def count_structures(n: int, min_hairpin: int = 3, max_interior: int = 30) -> float:
    return lib().orc_count_structures(n, min_hairpin, max_interior)


def mccaskill(model, seq) -> float:
    seq = np.ascontiguousarray(seq, dtype=np.uint8)
    m = make_model(model)
    return lib().orc_mccaskill(C.byref(m), len(seq), seq.ctypes.data_as(C.POINTER(C.c_uint8)))


class Tables:
    def __init__(self, handle, tt: TT, logZ: float):
        self.h, self.tt, self.logZ, self.n = handle, tt, logZ, tt.n

    def cell(self, which: int, i: int, j: int, shift: int = 0) -> np.ndarray:
        out = np.zeros(16 * 64 * 64)
        cnt = lib().orc_tables_cell(self.h, which, i, j, shift, _dp(out))
        return out[:cnt].copy()

    def logqext(self, j: int, c: int) -> float:
        return lib().orc_tables_logqext(self.h, j, c)

    def sample(self, J: int, seed: int):
        seq = np.zeros((J, self.n), dtype=np.uint8)
        pair = np.zeros((J, self.n), dtype=np.int32)
        lib().orc_sample(self.h, J, seed, seq.ctypes.data_as(C.POINTER(C.c_uint8)),
                         pair.ctypes.data_as(C.POINTER(C.c_int32)))
        return seq, pair

    def marginals(self):
        n = self.n
        bpp, base, codon = np.zeros((n, n)), np.zeros((n, 4)), np.zeros((n // 3, 64))
        rc = lib().orc_marginals(self.h, _dp(bpp), _dp(base), _dp(codon))
        if rc != 0:
            raise RuntimeError(f"orc_marginals rc={rc}")
        return bpp, base, codon

    def __del__(self):
        try:
            lib().orc_tables_free(self.h)
        except Exception:
            pass


def inside(model, tt: TT, nthreads: int = 0) -> Tables:
    m = make_model(model)
    h, logZ = C.c_void_p(), C.c_double()
    rc = lib().orc_inside(C.byref(m), tt.h, nthreads, C.byref(h), C.byref(logZ))
    if rc != 0:
        raise RuntimeError(f"orc_inside rc={rc}")
    return Tables(h, tt, logZ.value)


def uniform(seed, sample, kind, i, j) -> float:
    return lib().orc_uniform(seed, sample, kind, i, j)


NUC = "ACGU"


def seq_str(seq) -> str:
    return "".join(NUC[int(b)] for b in seq)


def dot_bracket(pair) -> str:
    return "".join("." if p < 0 else ("(" if p > k else ")") for k, p in enumerate(pair))


# ---- frequency matching, PAPER.md S4e (lines 751-771), Alg S4.6 "Naive iterative algorithm for frequency matching" -------------------
GENETIC_CODE = ("KNKNTTTTRSRSIIMI" "QHQHPPPPRRRRLLLL" "EDEDAAAAGGGGVVVV" "*Y*YSSSS*CWCLFLF")  # codon index 16 b0 + 4 b1 + b2, A,C,G,U = 0..3


def codon_marginals(tab: Tables) -> np.ndarray:
    """p_k(c) of eq 2.7 / 4.3 only (orc_marginals with the pair and base outputs switched off)."""
    codon = np.zeros((tab.n // 3, 64))
    rc = lib().orc_marginals(tab.h, None, None, _dp(codon))
    if rc != 0:
        raise RuntimeError(f"orc_marginals rc={rc}")
    return codon


def target_frequencies(aa: str, logf_star) -> np.ndarray:
    """b_* of Alg S4.6: "computed frequencies from U(psi) with applied multiplicative bonuses f_*" -- every residue picks a codon
    with probability proportional to its bonus, accumulated over the residues."""
    fs = np.exp(np.asarray(logf_star, dtype=np.float64))
    b = np.zeros(64)
    for a in aa:
        cod = [c for c in range(64) if GENETIC_CODE[c] == a]
        tot = sum(fs[c] for c in cod)
        for c in cod:
            b[c] += fs[c] / tot
    return b


def match_frequencies(model, aa: str, kind: int, logf_star, pair_logw=None, rtol: float = 2e-3, max_iter: int = 50, nthreads: int = 1):
    """Alg S4.6 line by line (naive iteration, no acceleration).  The update follows the prose of S4e step 2 ("multiply the current
    soft constraint bonus values by the ratio of desired frequencies divided by the achieved frequencies"): f <- f b_*/b; the update
    line of the printed pseudo-code has the ratio the other way round.  Requested frequencies equal to zero
    are left out (line 769).  Returns (log f, errors of the evaluated iterates)."""
    bstar = target_frequencies(aa, logf_star)
    act = bstar > 0
    logf = np.array(logf_star, dtype=np.float64)
    errs = []
    for _ in range(max_iter):
        tab = inside(model, TT.build(aa, kind, logf, pair_logw), nthreads)  # "Compute Q and free energy q_psi using bonuses f"
        b = codon_marginals(tab).sum(0)                               # "accumulated codon ... frequencies from these marginal probabilities"
        err = float(np.abs(np.log(b[act] / bstar[act])).max())        # "|| log(b / b_*) ||_inf"
        errs.append(err)
        if err < rtol:
            break
        logf[act] += np.log(bstar[act] / b[act])
    return logf, np.array(errs)


def mfe(model, tt: TT, nthreads: int = 0, brute: bool = False):
    """orc_mfe / orc_brute_force_min: (f_min in units of kT, seq uint8 [n], pair int32 [n]) -- PAPER.md eq 2.8."""
    m = make_model(model)
    f = C.c_double()
    seq = np.zeros(tt.n, dtype=np.uint8)
    pair = np.zeros(tt.n, dtype=np.int32)
    sp, pp = seq.ctypes.data_as(C.POINTER(C.c_uint8)), pair.ctypes.data_as(C.POINTER(C.c_int32))
    if brute:
        lib().orc_brute_force_min(C.byref(m), tt.h, C.byref(f), sp, pp)
    else:
        lib().orc_mfe(C.byref(m), tt.h, nthreads, C.byref(f), sp, pp)
    return f.value, seq, pair
