"""Build libcdz.so (the C-ABI CUDA library) and libcdz_peak.so (bench-only peak microbenchmarks) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
OUT = os.path.join(HERE, "libcdz.so")
OUT_PEAK = os.path.join(HERE, "libcdz_peak.so")
SOURCES = ["cdz_host.cu", "cdz_inside.cu", "cdz_cell.cu", "cdz_outside.cu", "cdz_usage.cu", "cdz_sample.cu",
           "cdz_eval.cu", "cdz_freq.cu", "cdz_mfe.cu", "cdz_tm.cu"]
PEAK_SOURCES = ["cdz_peak.cu"]  # not part of the product ABI: register-resident issue-rate loops for bench.py's roofline
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "--extended-lambda",
]


def _headers():
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    d.append(os.path.join(HERE, "..", "include", "cdz.h"))
    return d


def _compile(src: str, extra, verbose: bool) -> str:
    obj = os.path.join(OBJ, os.path.basename(src) + ".o")
    deps = [src] + _headers()
    if os.path.exists(obj) and all(os.path.getmtime(obj) >= os.path.getmtime(d) for d in deps):
        return obj
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
    subprocess.run(cmd, check=True)
    return obj


def _link(out: str, sources, force: bool, verbose: bool) -> str:
    srcs = [os.path.join(CSRC, s) for s in sources if os.path.exists(os.path.join(CSRC, s))]
    extra = os.environ.get("CDZ_NVCC_EXTRA", "").split()  # development only (e.g. -DCDZ_PHASE_TIMING)
    os.makedirs(OBJ, exist_ok=True)
    if force or extra:
        for s in srcs:
            o = os.path.join(OBJ, os.path.basename(s) + ".o")
            if os.path.exists(o):
                os.remove(o)
    with ThreadPoolExecutor(max_workers=min(8, len(srcs))) as ex:
        objs = list(ex.map(lambda s: _compile(s, extra, verbose), srcs))
    if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(o) for o in objs):
        return out
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-shared", "-o", out] + objs + ["-lcudart"], check=True)
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    _link(OUT_PEAK, PEAK_SOURCES, force, verbose)
    return _link(OUT, SOURCES, force, verbose)


if __name__ == "__main__":
    import sys

    print(build(force=True, verbose="-v" in sys.argv))
