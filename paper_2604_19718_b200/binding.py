"""Thin ctypes binding of libcdz.so (include/cdz.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of csrc/; torch is used for device
memory (workspace, outputs) and streams.  There is no CPU fallback: if the shared library
is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcdz.so")

TT_SINGLE_CODON, TT_CODON_PAIR = 0, 1
FP64, FP32_SCALED = 0, 1
NOALLOC_STACK_ITEMS = 400000  # CDZ_NOALLOC_STACK_ITEMS of include/cdz.h (limit of cdz_sample_noalloc)

EXPORTS = [
    "cdz_last_error", "cdz_version", "cdz_model_create", "cdz_model_destroy", "cdz_tt_build", "cdz_tt_build_pos",
    "cdz_tt_from_operators", "cdz_tt_destroy", "cdz_tt_length", "cdz_tt_describe", "cdz_workspace_bytes",
    "cdz_inside", "cdz_inside_batch", "cdz_inside_rerun", "cdz_inside_rerun_batch", "cdz_tables_logz",
    "cdz_tables_info", "cdz_tables_destroy", "cdz_tables_cell", "cdz_tables_logqext", "cdz_sample", "cdz_sample_noalloc",
    "cdz_debug_set_rescale_start", "cdz_eval_sequences", "cdz_match_frequencies", "cdz_mfe", "cdz_marginals", "cdz_marginals_workspace_bytes", "cdz_marginals_status", "cdz_run_host", "cdz_set_profiling", "cdz_profile",
    "cdz_tm_workspace_bytes", "cdz_tm_inside", "cdz_tm_block", "cdz_tm_sample",
]


class CdzError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"cdz error {code}: {msg}")
        self.code = code


class NNParams(C.Structure):
    _fields_ = [
        ("temperature_K", C.c_double), ("stack", C.c_double * 36), ("tmm", C.c_double * 96),
        ("hairpin_a", C.c_double), ("hairpin_b", C.c_double), ("hairpin_l0", C.c_double),
        ("bulge_init", C.c_double * 31), ("interior_init", C.c_double * 31),
        ("ml_a", C.c_double), ("ml_b", C.c_double), ("ml_c", C.c_double),
        ("max_interior", C.c_int32), ("min_hairpin", C.c_int32), ("allow_all_pairs", C.c_int32),
    ]


class Op(C.Structure):
    _fields_ = [("a", C.c_int32), ("b", C.c_int32), ("c", C.c_int32), ("x", C.c_double)]


class Info(C.Structure):
    _fields_ = [
        ("n", C.c_int32), ("sigma_bar", C.c_int32), ("n_left_states", C.c_int32), ("n_right_states", C.c_int32),
        ("precision", C.c_int32), ("n_rescales", C.c_int32), ("n_cc", C.c_double), ("n_loop", C.c_double),
        ("split_mac", C.c_double), ("table_bytes", C.c_double), ("bytes_per_cell", C.c_double),
        ("log_scale", C.c_double), ("inside_ms", C.c_double),
    ]


class TMParams(C.Structure):
    _fields_ = [("gamma", C.c_int32), ("xi", C.c_int32), ("min_hairpin", C.c_int32),
                ("V", C.POINTER(C.c_double)), ("B", C.POINTER(C.c_double)), ("S", C.POINTER(C.c_double))]


class TMInfo(C.Structure):
    _fields_ = [("device_ms", C.c_double), ("gemm_ms", C.c_double), ("block_ms", C.c_double), ("gemm_flop", C.c_double),
                ("table_bytes", C.c_double), ("launches", C.c_int64), ("gemm_launches", C.c_int64),
                ("S", C.c_int32), ("NB", C.c_int32), ("scale_rate", C.c_double)]


_lib = None


def lib():
    """Load libcdz.so; fails loudly if it has not been built (python -m paper_2604_19718_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python paper_2604_19718_b200/build.py` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    L.cdz_last_error.restype = C.c_char_p
    L.cdz_model_create.argtypes = [C.POINTER(NNParams), C.POINTER(vp)]
    L.cdz_model_destroy.argtypes = [vp]
    L.cdz_model_destroy.restype = None
    L.cdz_tt_build.argtypes = [C.c_char_p, C.c_int, C.c_int, dp, dp, C.POINTER(vp)]
    L.cdz_tt_build_pos.argtypes = [C.c_char_p, C.c_int, C.c_int, dp, dp, C.POINTER(vp)]
    L.cdz_tt_from_operators.argtypes = [C.c_int, C.POINTER(C.c_int32), C.POINTER(Op), C.POINTER(vp)]
    L.cdz_tt_destroy.argtypes = [vp]
    L.cdz_tt_destroy.restype = None
    L.cdz_tt_length.argtypes = [vp]
    L.cdz_tt_describe.argtypes = [vp, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.cdz_workspace_bytes.argtypes = [vp, C.c_int, C.POINTER(C.c_size_t)]
    L.cdz_inside.argtypes = [vp, vp, C.c_int, vp, C.c_size_t, vp, C.POINTER(vp), dp]
    L.cdz_inside_batch.argtypes = [vp, C.POINTER(vp), C.c_int, C.c_int, C.POINTER(vp), C.POINTER(C.c_size_t), vp,
                                   C.POINTER(vp), dp]
    L.cdz_inside_rerun.argtypes = [vp, vp]
    L.cdz_inside_rerun_batch.argtypes = [C.POINTER(vp), C.c_int, vp]
    L.cdz_tables_logz.argtypes = [vp, dp]
    L.cdz_tables_info.argtypes = [vp, C.POINTER(Info)]
    L.cdz_tables_destroy.argtypes = [vp]
    L.cdz_tables_destroy.restype = None
    L.cdz_set_profiling.argtypes = [vp, C.c_int]
    L.cdz_debug_set_rescale_start.argtypes = [vp, C.c_int]
    L.cdz_profile.argtypes = [vp, dp, C.POINTER(C.c_int64)]
    L.cdz_tables_cell.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, C.POINTER(C.c_int)]
    L.cdz_tables_logqext.argtypes = [vp, C.c_int, C.c_int, dp]
    L.cdz_sample.argtypes = [vp, C.c_int, C.c_uint64, vp, vp, vp]
    L.cdz_sample_noalloc.argtypes = [vp, C.c_int, C.c_uint64, vp, vp, vp]
    L.cdz_marginals.argtypes = [vp, vp, C.c_size_t, vp, vp, vp, vp]
    L.cdz_marginals_workspace_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    L.cdz_marginals_status.argtypes = [vp]
    L.cdz_eval_sequences.argtypes = [vp, vp, C.c_int, C.c_int, vp, C.c_int, dp, dp, dp, vp]
    L.cdz_match_frequencies.argtypes = [vp, C.c_char_p, C.c_int, C.c_int, dp, dp, C.c_double, C.c_int, C.c_int, dp, dp,
                                        C.POINTER(C.c_int), vp]
    L.cdz_mfe.argtypes = [vp, vp, vp, C.c_size_t, vp, dp, vp, vp]
    L.cdz_run_host.argtypes = [vp, C.c_int, C.c_uint64, vp, vp, dp, vp]
    L.cdz_tm_workspace_bytes.argtypes = [C.POINTER(TMParams), vp, C.POINTER(C.c_size_t)]
    L.cdz_tm_inside.argtypes = [C.POINTER(TMParams), vp, vp, C.c_size_t, vp, dp, C.POINTER(TMInfo)]
    L.cdz_tm_sample.argtypes = [C.POINTER(TMParams), vp, vp, C.c_int, C.c_uint64, vp, vp, vp]
    L.cdz_tm_block.argtypes = [C.POINTER(TMParams), vp, vp, C.c_double, C.c_int, C.c_int, C.c_int, dp, C.POINTER(C.c_int)]
    _lib = L
    return L


def _check(rc):
    if rc < 0:
        raise CdzError(rc, lib().cdz_last_error().decode())
    return rc


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _stream_ptr(stream):
    if stream is None:
        import torch

        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(getattr(stream, "cuda_stream", stream))


class Model:
    """cdz_model_create / cdz_model_destroy."""

    def __init__(self, m):
        p = NNParams()
        p.temperature_K = float(m.temperature_K)
        p.stack[:] = [float(v) for v in np.asarray(m.stack, dtype=np.float64).reshape(-1)]
        p.tmm[:] = [float(v) for v in np.asarray(m.tmm, dtype=np.float64).reshape(-1)]
        p.hairpin_a, p.hairpin_b, p.hairpin_l0 = float(m.hairpin_a), float(m.hairpin_b), float(m.hairpin_l0)
        p.bulge_init[:] = [float(v) for v in np.asarray(m.bulge_init, dtype=np.float64)]
        p.interior_init[:] = [float(v) for v in np.asarray(m.interior_init, dtype=np.float64)]
        p.ml_a, p.ml_b, p.ml_c = float(m.ml_a), float(m.ml_b), float(m.ml_c)
        p.max_interior, p.min_hairpin, p.allow_all_pairs = int(m.max_interior), int(m.min_hairpin), int(m.allow_all_pairs)
        self.h = C.c_void_p()
        _check(lib().cdz_model_create(C.byref(p), C.byref(self.h)))

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.cdz_model_destroy(self.h)
            self.h = None


class TensorTrain:
    """cdz_tt_build / cdz_tt_from_operators / cdz_tt_destroy."""

    def __init__(self, handle):
        self.h = handle
        self.n = lib().cdz_tt_length(handle)

    @classmethod
    def build(cls, aa: str, kind: int, codon_logw=None, pair_logw=None):
        """codon_logw: [64] (cdz_tt_build) or [L][64] per residue (cdz_tt_build_pos)."""
        cw = np.ascontiguousarray(codon_logw, dtype=np.float64) if codon_logw is not None else None
        pw = np.ascontiguousarray(pair_logw, dtype=np.float64).reshape(-1) if pair_logw is not None else None
        h = C.c_void_p()
        if cw is not None and cw.ndim == 2:
            if cw.shape != (len(aa), 64):
                raise ValueError("per-position codon weights must have shape [L][64]")
            _check(lib().cdz_tt_build_pos(aa.encode(), len(aa), kind, _dp(cw.reshape(-1)), _dp(pw), C.byref(h)))
        else:
            _check(lib().cdz_tt_build(aa.encode(), len(aa), kind, _dp(cw), _dp(pw), C.byref(h)))
        return cls(h)

    @classmethod
    def from_operators(cls, ops_per_pos):
        n = len(ops_per_pos)
        counts = (C.c_int32 * n)(*[len(o) for o in ops_per_pos])
        flat = [o for pos in ops_per_pos for o in pos]
        arr = (Op * max(1, len(flat)))()
        for k, (a, b, c, x) in enumerate(flat):
            arr[k] = Op(a, b, c, x)
        h = C.c_void_p()
        _check(lib().cdz_tt_from_operators(n, counts, arr, C.byref(h)))
        return cls(h)

    def describe(self):
        sigma = (C.c_int32 * (self.n + 1))()
        counts = (C.c_int32 * self.n)()
        nops = _check(lib().cdz_tt_describe(self.h, sigma, counts))
        return list(sigma), list(counts), nops

    def workspace_bytes(self, precision=FP64) -> int:
        b = C.c_size_t()
        _check(lib().cdz_workspace_bytes(self.h, precision, C.byref(b)))
        return b.value

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.cdz_tt_destroy(self.h)
            self.h = None


class Tables:
    """Handle returned by inside(); owns the torch workspace that backs the device tables."""

    def __init__(self, handle, model, tt, workspace):
        self.h, self.model, self.tt, self.workspace, self.n = handle, model, tt, workspace, tt.n

    def logz(self) -> float:
        v = C.c_double()
        _check(lib().cdz_tables_logz(self.h, C.byref(v)))
        return v.value

    def rerun(self, stream=None):
        _check(lib().cdz_inside_rerun(self.h, _stream_ptr(stream)))

    def info(self) -> dict:
        i = Info()
        _check(lib().cdz_tables_info(self.h, C.byref(i)))
        return {k: getattr(i, k) for k, _ in Info._fields_}

    def set_rescale_start(self, first: int):
        _check(lib().cdz_debug_set_rescale_start(self.h, first))

    def set_profiling(self, on: bool):
        _check(lib().cdz_set_profiling(self.h, 1 if on else 0))

    def profile(self) -> dict:
        """cdz_profile: per-kernel-class device ms and launch counts of the last pass."""
        ms = (C.c_double * 8)()
        ln = (C.c_int64 * 8)()
        _check(lib().cdz_profile(self.h, ms, ln))
        names = ["gemm", "block", "rescale", "exterior", "init", "sample", "c6", "c7"]
        return {"ms": dict(zip(names, list(ms))), "launches": dict(zip(names, list(ln)))}

    def cell(self, which, i, j):
        out = np.zeros(16 * 64)
        sh = C.c_int()
        cnt = _check(lib().cdz_tables_cell(self.h, which, i, j, _dp(out), C.byref(sh)))
        return out[:cnt].copy(), sh.value

    def logqext(self, j, c) -> float:
        v = C.c_double()
        _check(lib().cdz_tables_logqext(self.h, j, c, C.byref(v)))
        return v.value

    def sample(self, J: int, seed: int, stream=None):
        """cdz_sample: returns (seq uint8 [J,n], pair int32 [J,n]) as CUDA tensors."""
        import torch

        seq = torch.empty((J, self.n), dtype=torch.uint8, device="cuda")
        pair = torch.empty((J, self.n), dtype=torch.int32, device="cuda")
        _check(lib().cdz_sample(self.h, J, seed, C.c_void_p(seq.data_ptr()), C.c_void_p(pair.data_ptr()),
                                _stream_ptr(stream)))
        return seq, pair

    def sample_noalloc(self, J: int, seed: int, seq, pair, stream=None):
        """cdz_sample_noalloc: writes into the caller's CUDA tensors seq uint8 [J,n] and pair int32 [J,n]; allocates nothing."""
        _check(lib().cdz_sample_noalloc(self.h, J, seed, C.c_void_p(seq.data_ptr()), C.c_void_p(pair.data_ptr()),
                                        _stream_ptr(stream)))

    def marginals(self, stream=None, bpp=True, base=True, codon=True, own_workspace=True):
        """cdz_marginals: (bpp [n][n], base [n][4], codon [L][64]) as CUDA tensors (None where not requested), by the outside pass.
        The workspace is a torch tensor unless own_workspace=False (then the library uses the stream-ordered allocator).
        cdz_marginals_status is called before returning (it synchronises the stream)."""
        import torch

        n = self.n
        o_bpp = torch.empty((n, n), dtype=torch.float64, device="cuda") if bpp else None
        o_base = torch.empty((n, 4), dtype=torch.float64, device="cuda") if base else None
        o_codon = torch.empty((n // 3, 64), dtype=torch.float64, device="cuda") if codon else None
        ws, nb = None, 0
        if own_workspace:
            b = C.c_size_t()
            _check(lib().cdz_marginals_workspace_bytes(self.h, C.byref(b)))
            nb = b.value
            ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
        ptr = lambda x: C.c_void_p(x.data_ptr()) if x is not None else None  # noqa: E731
        _check(lib().cdz_marginals(self.h, ptr(ws), nb, ptr(o_bpp), ptr(o_base), ptr(o_codon), _stream_ptr(stream)))
        _check(lib().cdz_marginals_status(self.h))
        return o_bpp, o_base, o_codon

    def run_host(self, J: int, seed: int, seq_host=None, pair_host=None, stream=None) -> float:
        """cdz_run_host: host buffers in / out (pinned torch tensors or numpy arrays), returns log Z."""
        v = C.c_double()
        sp = C.c_void_p(seq_host.data_ptr()) if seq_host is not None else None
        pp = C.c_void_p(pair_host.data_ptr()) if pair_host is not None else None
        _check(lib().cdz_run_host(self.h, J, seed, sp, pp, C.byref(v), _stream_ptr(stream)))
        return v.value

    def destroy(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.cdz_tables_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        self.destroy()


def _alloc_workspace(tt, precision):
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: paper_2604_19718_b200 has no CPU fallback")
    nbytes = tt.workspace_bytes(precision)
    return torch.empty(nbytes, dtype=torch.uint8, device="cuda")


def inside(model: Model, tt: TensorTrain, precision=FP64, stream=None, sync=True):
    """cdz_inside: returns (Tables, logZ or None)."""
    ws = _alloc_workspace(tt, precision)
    h, lz = C.c_void_p(), C.c_double()
    _check(lib().cdz_inside(model.h, tt.h, precision, C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(stream),
                            C.byref(h), C.byref(lz) if sync else None))
    return Tables(h, model, tt, ws), (lz.value if sync else None)


def inside_batch(model: Model, tts, precision=FP64, stream=None):
    """cdz_inside_batch: returns ([Tables], [logZ])."""
    B = len(tts)
    wss = [_alloc_workspace(t, precision) for t in tts]
    tt_arr = (C.c_void_p * B)(*[t.h for t in tts])
    ws_arr = (C.c_void_p * B)(*[w.data_ptr() for w in wss])
    wb_arr = (C.c_size_t * B)(*[w.numel() for w in wss])
    out = (C.c_void_p * B)()
    lz = (C.c_double * B)()
    _check(lib().cdz_inside_batch(model.h, tt_arr, B, precision, ws_arr, wb_arr, _stream_ptr(stream), out, lz))
    return [Tables(C.c_void_p(out[b]), model, tts[b], wss[b]) for b in range(B)], list(lz)


def inside_rerun_batch(tables, stream=None):
    B = len(tables)
    arr = (C.c_void_p * B)(*[t.h.value for t in tables])
    _check(lib().cdz_inside_rerun_batch(arr, B, _stream_ptr(stream)))


def eval_sequences(model: Model, design: TensorTrain | None, seqs, want_unpaired=False, max_batch=0, stream=None):
    """cdz_eval_sequences: seqs [J][n] uint8 (numpy or CPU tensor).  Returns (logZ [J], logW [J] or None, unpaired [J][n] or None)."""
    seqs = np.ascontiguousarray(np.asarray(seqs), dtype=np.uint8)
    J, n = seqs.shape
    lz = np.zeros(J)
    lw = np.zeros(J) if design is not None else None
    un = np.zeros((J, n)) if want_unpaired else None
    _check(lib().cdz_eval_sequences(model.h, design.h if design is not None else None, n, J,
                                    seqs.ctypes.data_as(C.c_void_p), max_batch, _dp(lz), _dp(lw), _dp(un), _stream_ptr(stream)))
    return lz, lw, un


def match_frequencies(model: Model, aa: str, kind: int, logf_star, pair_logw=None, rtol=2e-3, max_iter=50, anderson=True, stream=None):
    """cdz_match_frequencies (Alg S4.6): returns (logf [64], errors of the evaluated iterates)."""
    fs = np.ascontiguousarray(logf_star, dtype=np.float64)
    pw = np.ascontiguousarray(pair_logw, dtype=np.float64).reshape(-1) if pair_logw is not None else None
    out = np.zeros(64)
    errs = np.zeros(max_iter)
    nit = C.c_int()
    _check(lib().cdz_match_frequencies(model.h, aa.encode(), len(aa), kind, _dp(fs), _dp(pw), rtol, max_iter, 1 if anderson else 0,
                                       _dp(out), _dp(errs), C.byref(nit), _stream_ptr(stream)))
    return out, errs[:nit.value].copy()


def mfe(model: Model, tt: TensorTrain, traceback=True, stream=None):
    """cdz_mfe: (f_min in units of kT, seq uint8 [n] CUDA tensor or None, pair int32 [n] CUDA tensor or None) -- PAPER.md eq 2.8."""
    import torch

    ws = _alloc_workspace(tt, FP64)
    f = C.c_double()
    seq = torch.empty(tt.n, dtype=torch.uint8, device="cuda") if traceback else None
    pair = torch.empty(tt.n, dtype=torch.int32, device="cuda") if traceback else None
    _check(lib().cdz_mfe(model.h, tt.h, C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(stream), C.byref(f),
                         C.c_void_p(seq.data_ptr()) if traceback else None, C.c_void_p(pair.data_ptr()) if traceback else None))
    return f.value, seq, pair


class TensorModelPass:
    """cdz_tm_inside: the paper's tensor-model recursion (eqs 3.5-3.8) over a tensor train; keeps the workspace so that blocks can be read back."""

    def __init__(self, tm, tt: TensorTrain, stream=None):
        import torch

        self._V = np.ascontiguousarray(tm.V, dtype=np.float64)
        self._B = np.ascontiguousarray(tm.B, dtype=np.float64)
        self._S = np.ascontiguousarray(tm.S, dtype=np.float64)
        self.p = TMParams(int(tm.gamma), int(tm.xi), int(tm.min_hairpin), _dp(self._V), _dp(self._B), _dp(self._S))
        self.tt = tt
        nb = C.c_size_t()
        _check(lib().cdz_tm_workspace_bytes(C.byref(self.p), tt.h, C.byref(nb)))
        self.ws = torch.empty(nb.value, dtype=torch.uint8, device="cuda")
        self.info = TMInfo()
        lz = C.c_double()
        _check(lib().cdz_tm_inside(C.byref(self.p), tt.h, C.c_void_p(self.ws.data_ptr()), nb.value, _stream_ptr(stream), C.byref(lz),
                                   C.byref(self.info)))
        self.logZ = lz.value

    def rerun(self, stream=None):
        lz = C.c_double()
        _check(lib().cdz_tm_inside(C.byref(self.p), self.tt.h, C.c_void_p(self.ws.data_ptr()), self.ws.numel(), _stream_ptr(stream),
                                   C.byref(lz), C.byref(self.info)))
        self.logZ = lz.value
        return lz.value

    def block(self, which: int, i: int, j: int):
        """(values as stored, shift): true block = values * 2**shift.  which 0: Q_{i,j} upper, 1: Q_{j,i} lower."""
        out = np.zeros(32 * 32)
        sh = C.c_int()
        cnt = _check(lib().cdz_tm_block(C.byref(self.p), self.tt.h, C.c_void_p(self.ws.data_ptr()), self.info.scale_rate, which, i, j,
                                        _dp(out), C.byref(sh)))
        return out[:cnt].copy(), sh.value

    def sample(self, J: int, seed: int, stream=None):
        """cdz_tm_sample: (seq uint8 [J][n], pair int32 [J][n]) CUDA tensors."""
        import torch

        n = self.tt.n
        seq = torch.empty((J, n), dtype=torch.uint8, device="cuda")
        pair = torch.empty((J, n), dtype=torch.int32, device="cuda")
        _check(lib().cdz_tm_sample(C.byref(self.p), self.tt.h, C.c_void_p(self.ws.data_ptr()), J, seed, C.c_void_p(seq.data_ptr()),
                                   C.c_void_p(pair.data_ptr()), _stream_ptr(stream)))
        return seq, pair
