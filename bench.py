#!/usr/bin/env python
"""bench.py -- headline measurement of the codon-design inside pass on B200 (one JSON line on stdout).

A "step" is one pass of the whole hot path over one synthetic design: the inside pass
(stretch products, closed cells, split-point GEMM, per-position rescaling, exterior, log Z) followed by the
stochastic traceback of the config's sample count.  The tensor train and the loop Boltzmann tables are built on the
host before the timed region (8a-1/8a-2 are O(n) host work) and are resident in HBM when it starts.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cdz|reference] [--config C] [--L aa]

Workload at N=1: BASELINE.json configs[3], the 5000-aa (15000-nt) design the metric is quoted on.
N>1 (torchrun): replicas only -- one design does not shard; every rank runs the same
design independently, no data-path collective, `value` = N x units / max-over-ranks time ("scaling": "weak").
--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "DP-cell-contractions/s per design (N_cc + N_loop terms of the inside pass / step time)"
UNIT = "cell-contractions/s"
SAMPLES = {1: 1000, 2: 0, 3: 0, 4: 100, 5: 256}
WORKLOADS = {
    1: "configs[0]: 20-aa protein, single-codon TT, fp64, 1000 samples",
    2: "configs[1]: 300-aa protein, codon-pair TT, fp64",
    3: "configs[2]: 1000-aa protein (3000 nt), codon-pair TT, fp32-scaled split-point contraction (3xTF32, fp64 tables)",
    4: "configs[3]: 5000-aa protein (15000 nt), single-codon TT, codon weights, fp64 inside pass + 100 samples",
    5: "configs[4]: 150-aa protein, codon-pair TT, fp64, 256 samples (one item of the batch)",
}


def counts(n: int, min_hairpin: int = 3, max_interior: int = 30):
    """N_cc and N_loop of SURVEY.md 8(d) (closed forms, independent of the library)."""
    mh1 = min_hairpin + 1
    ncc = nloop = 0
    per_d = {}
    for d in range(n):
        ncc += (n - d) * max(0, d - 2 * mh1)
        key = min(d, 2 * max_interior + 16)
        if key not in per_d:
            per_d[key] = sum(1 for l1 in range(max_interior + 1) for l2 in range(max_interior + 1 - l1)
                             if d - 2 - l1 - l2 >= mh1)
        nloop += (n - d) * per_d[key]
    return float(ncc), float(nloop)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(r) > 2 + k and r[2 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


_peak_lib = None


def peak_lib():
    """libcdz_peak.so: register-resident issue-rate loops and latency probes (bench only, not part of the product ABI)."""
    global _peak_lib
    if _peak_lib is None:
        import ctypes as C

        _peak_lib = C.CDLL(os.path.join(ROOT, "paper_2604_19718_b200", "libcdz_peak.so"))
        _peak_lib.cdz_peak_measure.argtypes = [C.c_int, C.POINTER(C.c_double)]
        _peak_lib.cdz_peak_launch_us.argtypes = [C.c_int, C.POINTER(C.c_double)]
        _peak_lib.cdz_peak_barrier_us.argtypes = [C.c_int, C.POINTER(C.c_double)]
    return _peak_lib


def measure_peak(kind: int) -> float:
    """0 fp64 FMA, 1 fp64 mma.sync m8n8k4, 2 fp32 FMA (TFLOP/s)."""
    import ctypes as C

    v = C.c_double()
    rc = peak_lib().cdz_peak_measure(kind, C.byref(v))
    if rc != 0:
        raise RuntimeError(f"cdz_peak_measure rc={rc}")
    return v.value


def reduce_max(value: float, device="cpu") -> float:
    """Max over ranks of a per-rank time (the only collective besides the barrier: replicas share no data)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, world: int, ms_max: float) -> float:
    """Replicas only: every rank processes the same units, the job takes the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)


def oracle_sample(cfg: int, L_sample: int):
    """Time the CPU oracle's inside pass, as it stands, on the first L_sample residues of the workload."""
    from oracle import oracle as O
    from paper_2604_19718_b200 import inputs as I

    d = I.design(cfg, 0, L_sample)
    tt = O.TT.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    t0 = time.perf_counter()
    tab = O.inside(I.nn_model(), tt, 0)
    dt = time.perf_counter() - t0
    ncc, nloop = counts(d.n)
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    return dict(value=(ncc + nloop) / dt, seconds=dt, cores=cores, n=d.n, logZ=tab.logZ,
                sample=f"oracle inside pass (orc_inside, OpenMP over the cells of a diagonal) on the first {L_sample} aa "
                       f"({d.n} nt) of the workload's design: {ncc + nloop:.3e} cell-contractions in {dt:.1f} s")


ORACLE_L = {1: 20, 2: 60, 3: 60, 4: 100, 5: 60}  # residues of the bounded oracle sample (config 1: the whole design)


def oracle_full_size(cfg: int, sample: dict):
    """The oracle on the WHOLE workload: the stored run of tests/golden/oracle_logz.txt where one exists (measured once on the
    8-core build box by tests/golden/make_golden.py, oracle only), otherwise an extrapolation from the live sample, labelled."""
    path = os.path.join(ROOT, "tests", "golden", "oracle_logz.txt")
    full_L = {1: 20, 2: 300, 3: 1000, 4: 5000, 5: 150}[cfg]
    try:
        for ln in open(path):
            f = ln.split()
            if f and f[0] == str(cfg) and int(f[2]) == full_L:
                n = int(f[3])
                ncc, nloop = counts(n)
                sec = max(float(f[5]), 0.5)
                return {"kind": "stored", "seconds": sec, "cores": 8, "value": (ncc + nloop) / sec, "unit": UNIT,
                        "note": "whole design, plain long-double recursion, measured on the 8-core build box (tests/golden/oracle_logz.txt)"}
    except OSError:
        pass
    n_full = 3 * full_L
    ncc, nloop = counts(n_full)
    ncs, nls = counts(sample["n"])
    # loop terms scale with their count; the split-point sum with N_cc (the sample's cost is dominated by the loop terms)
    sec = sample["seconds"] * ((nloop + ncc) / max(nls + ncs, 1.0))
    return {"kind": "EXTRAPOLATED", "seconds": sec, "cores": sample["cores"], "value": (ncc + nloop) / sec, "unit": UNIT,
            "note": "EXTRAPOLATED from the live sample by the ratio of cell-contraction counts (the plain oracle cannot hold a "
                    f"{n_full}-nt design: long-double range and hours of CPU time); not a measurement"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    L_sample = args.oracle_L or ORACLE_L[cfg]
    vals = []
    for _ in range(args.warmup):
        pass  # the oracle has no warm state; warm-up steps are no-ops
    last = None
    for _ in range(max(1, args.steps)):
        last = oracle_sample(cfg, L_sample)
        vals.append(last)
    tot_units = sum(v["value"] * v["seconds"] for v in vals)
    tot_s = sum(v["seconds"] for v in vals)
    value = tot_units / tot_s
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / len(vals),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 (long double oracle)",
        "data": "synthetic", "config": {"workload": WORKLOADS[cfg], "bounded_sample": last["sample"]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


def run_cdz(args):
    import torch
    import torch.distributed as dist

    from paper_2604_19718_b200 import binding as B
    from paper_2604_19718_b200 import build
    from paper_2604_19718_b200 import inputs as I

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()

    cfg = args.config
    d = I.design(cfg, 0, args.L)
    J = SAMPLES[cfg] if args.samples is None else args.samples
    model = B.Model(I.nn_model())
    tt = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    fp32 = (args.precision == "fp32") if args.precision else (cfg == 3)
    tab, logz0 = B.inside(model, tt, precision=B.FP32_SCALED if fp32 else B.FP64)  # allocation + first pass (untimed)
    n = d.n
    ncc, nloop = counts(n)
    units = ncc + nloop
    stream = torch.cuda.current_stream()
    seq = torch.empty((max(J, 1), n), dtype=torch.uint8, device="cuda")
    pair = torch.empty((max(J, 1), n), dtype=torch.int32, device="cuda")

    def step():
        tab.rerun(stream)
        if J > 0:
            B._check(B.lib().cdz_sample(tab.h, J, d.sample_seed, B.C.c_void_p(seq.data_ptr()),
                                        B.C.c_void_p(pair.data_ptr()), B._stream_ptr(stream)))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-timed region -------------------------------------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    prof_ms = {}
    prof_launches = {}
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clk = clocks.stop() if rank == 0 else None
    # per-kernel-class device times: ONE extra, untimed step with an event between consecutive launches (the timed steps above run
    # with profiling off, so no event records sit inside the timed region)
    tab.set_profiling(True)
    step()
    torch.cuda.synchronize()
    prof = tab.profile()
    prof_ms, prof_launches = prof["ms"], prof["launches"]
    tab.set_profiling(False)
    logz = tab.logz()
    info = tab.info()
    ms_step = reduce_max(ms_total, "cuda") / args.steps
    value = whole_job_value(units, world, ms_step)

    # ---- end to end through the C ABI with host buffers --------------------------------------------------------------
    seq_h = torch.empty((max(J, 1), n), dtype=torch.uint8).pin_memory()
    pair_h = torch.empty((max(J, 1), n), dtype=torch.int32).pin_memory()
    sigma, cnts, nops = tt.describe()
    h2d = nops * (5 + 8 * 2) + 4 * (5 * (n + 2)) + 8 * 2 * n * info_ms2(sigma) + 8 * (n + 1)
    d2h = (J * n * 5 if J > 0 else 0) + 8 * 4 + 4 * 4
    e2e_steps = max(1, min(args.steps, 3))
    tab.run_host(J, d.sample_seed, seq_h if J else None, pair_h if J else None, stream)  # warm-up
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        # the user's call sequence: build the tensor train from the protein and the weights (host, O(n)), then one host-buffer call
        # (operator lists and cores host -> device, inside pass, traceback, samples device -> host, log Z)
        tt_step = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
        lz_e2e = tab.run_host(J, d.sample_seed, seq_h if J else None, pair_h if J else None, stream)
        del tt_step
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    e2e_value = whole_job_value(units, world, 1e3 * reduce_max(e2e_s, "cuda"))

    # ---- optional: outside pass (base-pair probabilities) on the tables of the last inside pass; outside the timed step
    marg = None
    if args.marginals and rank == 0:
        tab.rerun(stream)
        bpp, base_m, codon_m = tab.marginals(stream)  # warm-up
        torch.cuda.synchronize()
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        m0.record(stream)
        bpp, base_m, codon_m = tab.marginals(stream)
        m1.record(stream)
        torch.cuda.synchronize()
        up = torch.triu(bpp, 1)
        marg = {"what": "cdz_marginals: outside / adjoint pass -> base-pair probabilities (eq 2.5), base (eq 2.6) and codon (eq 2.7) "
                        "marginals, DESIGN.md section 9",
                "ms": m0.elapsed_time(m1), "ratio_to_inside": m0.elapsed_time(m1) / info["inside_ms"], "gpu_launches": n + 7,
                "expected_pairs": float(up.sum()),
                "max_row_sum_error": float(((up + up.T).sum(1) + torch.diagonal(bpp) - 1.0).abs().max()),
                "max_base_sum_error": float((base_m.sum(1) - 1.0).abs().max()),
                "max_codon_sum_error": float((codon_m.sum(1) - 1.0).abs().max()),
                "note": "the unpaired diagonal and the base / codon marginals come from the operator usages, so none of the three sum "
                        "rules holds by construction; device time by CUDA events, workspace allocated by the caller beforehand "
                        "(allocation of the torch tensor inside the timed call)"}
        del bpp, base_m, codon_m, up

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel -----------------------------------------------------------------------------
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
    except OSError:
        pass
    dmma = measure_peak(1)
    dfma = measure_peak(0)
    ffma = measure_peak(2)
    bf16 = peaks.get("bf16_tflops")
    sbar_n = info["sigma_bar"] / n
    loop_mac = nloop * 2.0 * sbar_n ** 3
    cls = {k: v for k, v in prof_ms.items() if k in ("gemm", "block", "rescale", "exterior", "sample")}
    dominant = max(cls, key=cls.get) if cls else "gemm"
    gemm_ms, gemm_l = prof_ms.get("gemm", 0.0), prof_launches.get("gemm", 0)
    roof_gemm = None
    if gemm_ms > 0 and fp32:
        ach = 2.0 * info["split_mac"] / (gemm_ms * 1e-3) / 1e12
        roof_gemm = {"kernel": "gemm32_kernel (split-point contraction, 3xTF32 on mma.sync m16n8k8, fp32 accumulate, fp64 operands in HBM)",
                     "bound": "tensor", "achieved": ach, "peak": ffma, "unit": "TFLOP/s", "frac": ach / ffma, "traffic": None,
                     "launches": gemm_l, "avg_launch_ms": gemm_ms / max(gemm_l, 1),
                     "algorithmic_flop_per_step": 2.0 * info["split_mac"],
                     "peak_source": "in-run register-resident fp32 FMA loop (libcdz_peak.so): the vector fp32 rate is the bar an "
                                    "exact-to-fp32 contraction has to beat; the 3xTF32 split issues 3 MMAs per product",
                     "share_of_step": gemm_ms / ms_step}
    elif gemm_ms > 0:
        ach = 2.0 * info["split_mac"] / (gemm_ms * 1e-3) / 1e12
        roof_gemm = {"kernel": "gemm_kernel (split-point contraction, fp64 mma.sync m8n8k4)", "bound": "tensor",
                     "achieved": ach, "peak": dmma, "unit": "TFLOP/s", "frac": ach / dmma, "traffic": None,
                     "launches": gemm_l, "avg_launch_ms": gemm_ms / max(gemm_l, 1),
                     "algorithmic_flop_per_step": 2.0 * info["split_mac"],
                     "peak_source": "in-run register-resident mma.sync.m8n8k4.f64 loop (cdz_measure_peak); "
                                    "MEASURED_PEAKS.json has no fp64 entry; rule-derived alternative = bf16_tflops x "
                                    "45/2250 = %s" % (None if bf16 is None else round(bf16 * 45.0 / 2250.0, 2)),
                     "share_of_step": gemm_ms / ms_step}
    # dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed ncu summary of THIS source state only: the file
    # records a hash of the kernel sources; if the sources have changed since the capture the traffic is reported as null
    ncu_traffic = committed_traffic(cfg if not args.L else None)
    if roof_gemm:
        roof_gemm["traffic"] = ncu_traffic.get("gemm")
    block_ms, block_l = prof_ms.get("block", 0.0), prof_launches.get("block", 0)
    roof_block = None
    if block_ms > 0:
        ach = 2.0 * loop_mac / (block_ms * 1e-3) / 1e12
        roof_block = {"kernel": "cell_kernel (closed cells: hairpin/stack/bulge/interior<=30/multiloop closure, Qm1/Qml, in-block edge splits)",
                      "bound": "alu", "achieved": ach, "peak": dfma, "unit": "TFLOP/s", "frac": ach / dfma,
                      "traffic": ncu_traffic.get("block"), "launches": block_l, "avg_launch_ms": block_ms / max(block_l, 1),
                      "algorithmic_flop_per_step": 2.0 * loop_mac,
                      "note": "latency-bound, not ALU-bound: see latency_floor (DESIGN.md 8.1)",
                      "peak_source": "in-run register-resident fp64 FMA loop (cdz_measure_peak)",
                      "share_of_step": block_ms / ms_step}
    roofline = roof_block if dominant == "block" and roof_block else (roof_gemm or roof_block)

    # the third number: dependency-latency floor of the blocked wavefront = launches x (empty dependent launch) +
    # in-block anti-diagonal steps x barrier rounds per step x (one __syncthreads round of a 512-thread CTA), both measured here
    import ctypes as C

    t_launch, t_bar = C.c_double(), C.c_double()
    peak_lib().cdz_peak_launch_us(2000, C.byref(t_launch))
    peak_lib().cdz_peak_barrier_us(20000, C.byref(t_bar))
    sigma, _, _ = tt.describe()
    nb_blocks = int(prof_launches.get("block", 0))
    pos_per_block = (n + 1) / max(nb_blocks, 1)
    inblock_steps = nb_blocks * (2.0 * pos_per_block - 1.0)
    barriers_per_step = 6
    n_launch = sum(int(v) for k, v in prof_launches.items() if k != "sample")
    latency_floor = {"launches": n_launch, "t_launch_us": t_launch.value, "in_block_steps": inblock_steps,
                     "barrier_rounds_per_step": barriers_per_step, "t_barrier_round_us": t_bar.value,
                     "floor_ms": 1e-3 * (n_launch * t_launch.value + inblock_steps * barriers_per_step * t_bar.value),
                     "note": "lower bound from empty dependent launches and empty barrier rounds only; the measured step also waits "
                             "on dependent global / shared memory loads inside every round"}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        o = oracle_sample(cfg, args.oracle_L or ORACLE_L[cfg])
        cpu = {"value": o["value"], "unit": UNIT, "cores": o["cores"], "kind": "oracle", "sample": o["sample"],
               "full_size": oracle_full_size(cfg, o)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 contraction (3xTF32) + f64 tables" if fp32 else "f64",
        "data": "synthetic",
        "config": {"workload": WORKLOADS.get(cfg, f"config {cfg}") + (f" [L overridden to {args.L}]" if args.L else ""),
                   "n_nt": n, "sigma_bar": info["sigma_bar"], "samples_per_step": J, "parallelism": "replicas only",
                   "l2": "tables (%.1f GB) larger than L2; no flush needed" % (info["table_bytes"] / 1e9)
                   if info["table_bytes"] > 2.5e8 else "tables smaller than L2: warm-cache number",
                   "seed": d.seed, "nn_model_seed": 19718},
        "inside_ms": info["inside_ms"], "n_cc": ncc, "n_loop": nloop, "n_cc_per_s": ncc / (info["inside_ms"] * 1e-3),
        "split_mac": info["split_mac"], "logZ": logz, "table_bytes": info["table_bytes"],
        "bytes_per_cell": info["bytes_per_cell"], "n_rescales": info["n_rescales"],
        "kernel_ms": prof_ms, "kernel_launches": prof_launches,
        "gpu_launches": int(sum(prof_launches.values())) * args.steps,
        "roofline": roofline, "roofline_gemm": roof_gemm, "roofline_block": roof_block,
        "peaks": {"fp64_fma_tflops": dfma, "fp64_mma_tflops": dmma, "fp32_fma_tflops": ffma, "hbm_gbs": peaks.get("hbm_gbs"),
                  "bf16_tflops": bf16},
        "latency_floor": latency_floor,
        "cpu_baseline": cpu,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": 1e3 * e2e_s, "logZ": lz_e2e,
                "timed_region": "cdz_tt_build (host) + cdz_run_host: h2d of operator lists / cores, inside pass, traceback, d2h of "
                                "samples and log Z; the device workspace and the model handle are created once before it"},
        "clocks": clk,
    }
    if marg is not None:
        out["marginals"] = marg
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_batch(args):
    """configs[4]: B independent 150-aa designs (distinct seeds) advanced together by cdz_inside_batch, 256 samples each.
    Secondary measurement (small-design throughput); the default bench line is the 5000-aa design."""
    import torch

    from paper_2604_19718_b200 import binding as B
    from paper_2604_19718_b200 import build
    from paper_2604_19718_b200 import inputs as I

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU fallback)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    build.build()
    nb = args.batch
    J = SAMPLES[5] if args.samples is None else args.samples
    ds = [I.design(5, item, args.L) for item in range(nb)]
    model = B.Model(I.nn_model())
    tts = [B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw) for d in ds]
    tabs, lzs = B.inside_batch(model, tts)
    n = ds[0].n
    ncc, nloop = counts(n)
    units = nb * (ncc + nloop)
    stream = torch.cuda.current_stream()
    seq = torch.empty((nb, max(J, 1), n), dtype=torch.uint8, device="cuda")
    pair = torch.empty((nb, max(J, 1), n), dtype=torch.int32, device="cuda")

    side = [torch.cuda.Stream() for _ in range(min(16, nb))]  # the designs' tracebacks are independent: run them concurrently

    def step():
        B.inside_rerun_batch(tabs, stream)
        if J > 0:
            done = torch.cuda.Event()
            done.record(stream)
            for k, (tab, d) in enumerate(zip(tabs, ds)):
                st = side[k % len(side)]
                st.wait_event(done)
                B._check(B.lib().cdz_sample(tab.h, J, d.sample_seed, B.C.c_void_p(seq[k].data_ptr()),
                                            B.C.c_void_p(pair[k].data_ptr()), B._stream_ptr(st)))
            for st in side:
                stream.wait_stream(st)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    clocks = ClockSampler(0)
    clocks.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ev[0].record(stream)
    for _ in range(args.steps):
        B.inside_rerun_batch(tabs, stream)
    ev[1].record(stream)
    for _ in range(args.steps):
        step()
    ev[2].record(stream)
    torch.cuda.synchronize()
    inside_ms = ev[0].elapsed_time(ev[1]) / args.steps
    ms_step = ev[1].elapsed_time(ev[2]) / args.steps
    clk = clocks.stop()
    lz2 = [t.logz() for t in tabs]
    out = {
        "metric": METRIC, "value": units / (ms_step * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"configs[4]: batch of {nb} independent {n // 3}-aa proteins ({n} nt), codon-pair TT, fp64 inside pass "
                               f"+ {J} samples each, one batched launch sequence", "batch": nb, "n_nt": n, "samples_per_step": nb * J,
                   "l2": "tables of the batch smaller than L2 at small B: warm-cache number"},
        "inside_ms": inside_ms, "designs_per_s": nb / (ms_step * 1e-3), "logZ_first": lzs[0],
        "deterministic": lz2 == lzs, "clocks": clk,
    }
    print(json.dumps(out), flush=True)


def run_tensor_model(args):
    """Secondary measurement: the paper's own recursion -- tensor-based model (gamma, xi synthetic) x codon tensor train of a
    BASELINE design -- through cdz_tm_inside.  One step = one full call (pilot passes, table clear, all block diagonals, final trace)."""
    import time

    import torch

    from paper_2604_19718_b200 import binding as B
    from paper_2604_19718_b200 import build
    from paper_2604_19718_b200 import inputs as I

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU fallback)")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    build.build()
    cfg = args.config if args.config != 4 or args.L else 3  # default workload of this mode: configs[2], 1000 aa, codon-pair tensor train
    d = I.design(cfg, 0, args.L)
    tm = I.tensor_model(args.gamma, args.xi)
    tt = B.TensorTrain.build(d.aa, d.kind, d.codon_logw, d.pair_logw)
    run = B.TensorModelPass(tm, tt)
    for _ in range(max(args.warmup, 3) - 1):
        run.rerun()
    clocks = ClockSampler(0)
    clocks.start()
    dev, gemm, block, wall = [], [], [], []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        run.rerun()
        wall.append((time.perf_counter() - t0) * 1e3)
        dev.append(run.info.device_ms); gemm.append(run.info.gemm_ms); block.append(run.info.block_ms)
    # 100 exact samples from the tables of the last pass (cdz_tm_sample), device time by CUDA events on the launching stream
    nsmp = 100
    run.sample(nsmp, 1)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    seq, pair = run.sample(nsmp, d.sample_seed)
    ev1.record()
    torch.cuda.synchronize()
    sample_ms = ev0.elapsed_time(ev1)
    paired = float((pair >= 0).float().mean().item())
    clk = clocks.stop()
    ms, gms, bms, wms = (sum(v) / len(v) for v in (dev, gemm, block, wall))
    peak = measure_peak(1)
    i = run.info
    sig = tt.describe()[0]
    flat = args.gamma * sum(sig)
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import oracle as O
        from oracle import tensor_model as TM

        Ls = 16
        so, oo = O.TT.build(d.aa[:Ls], d.kind, d.codon_logw, d.pair_logw).get()
        t0 = time.perf_counter()
        TM.tm_inside(tm, so, oo)
        sec = time.perf_counter() - t0
        cpu = {"value": sec * 1e3, "unit": "ms", "cores": 1, "kind": "oracle",
               "sample": f"oracle/tensor_model.py tm_inside (plain numpy Alg S4.1) on the first {Ls} aa ({3 * Ls} nt) of the same design: {sec:.1f} s; "
                         "cost grows as n^3, not comparable with the full-size GPU time"}
    out = {
        "metric": "tensor-model partition function (PAPER.md eqs 3.5-3.8), device time of one full pass", "value": ms, "unit": "ms",
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"configs[{cfg - 1}] design ({len(d.aa)} aa, {d.n} nt, {'codon-pair' if d.kind else 'single-codon'} tensor train) under a "
                               f"synthetic tensor model gamma={args.gamma} xi={args.xi}", "n_nt": d.n, "flattened_dim": flat, "padded_dim": i.S,
                   "blocks": i.NB, "l2": f"tables ({i.table_bytes / 1e9:.1f} GB) larger than L2" if i.table_bytes > 126e6 else "tables fit L2"},
        "logZ": run.logZ, "scale_rate_bits_per_nt": i.scale_rate, "gemm_ms": gms, "block_ms": bms, "gpu_launches": int(i.launches),
        "samples": {"n": nsmp, "ms": sample_ms, "paired_fraction": paired, "what": "cdz_tm_sample: exact (sequence, structure) samples by stochastic traceback of the tables of the pass"},
        "roofline": {"kernel": "tm_gemm_kernel (k-sum over finished blocks, fp64 mma.sync m8n8k4 tiles shared with the inside pass)",
                     "bound": "tensor", "achieved": i.gemm_flop / (gms * 1e-3) / 1e12 if gms > 0 else None, "peak": peak, "unit": "TFLOP/s",
                     "frac": (i.gemm_flop / (gms * 1e-3) / 1e12 / peak) if gms > 0 else None, "traffic": None,
                     "launches": int(i.gemm_launches), "flop_per_step": i.gemm_flop,
                     "note": "FLOP of the 64-padded tiles; the unpadded flattened dimension is config.flattened_dim",
                     "peak_source": "in-run register-resident mma.sync.m8n8k4.f64 loop (libcdz_peak.so)", "share_of_step": gms / ms},
        "cpu_baseline": cpu,
        "e2e": {"value": wms, "unit": "ms", "h2d_bytes_per_step": int(8 * 4 * d.n * max(sig) ** 2), "d2h_bytes_per_step": 8,
                "timed_region": "host wall clock of cdz_tm_inside: dense cores built on the host and copied, two pilot passes, the full pass, log Z read back"},
        "clocks": clk,
    }
    print(json.dumps(out), flush=True)


def kernel_source_hash() -> str:
    import hashlib

    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2604_19718_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".h", ".cuh")):
            h.update(open(os.path.join(csrc, name), "rb").read())
    return h.hexdigest()[:16]


def committed_traffic(cfg):
    """profiles/traffic.json.txt: {"source_hash": "...", "config": 4, "gemm": bytes per launch, "block": bytes per launch, "from": "..."}.
    Only used when it was captured from exactly these kernel sources and this config; otherwise {} (traffic: null)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json.txt")) as f:
            rec = json.load(f)
    except (OSError, ValueError):
        return {}
    if rec.get("source_hash") != kernel_source_hash() or rec.get("config") != cfg:
        return {}
    return rec


def info_ms2(sigma) -> int:
    ms = max(sigma)
    return ms * ms


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cdz", choices=["cdz", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--precision", default=None, choices=["fp64", "fp32"], help="default: fp32 for config 3, fp64 otherwise")
    ap.add_argument("--L", type=int, default=None, help="override the protein length (development only)")
    ap.add_argument("--samples", type=int, default=None)
    ap.add_argument("--oracle-L", type=int, default=None, dest="oracle_L")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--marginals", action="store_true", help="also time cdz_marginals (base-pair probabilities) after the timed steps")
    ap.add_argument("--batch", type=int, default=0, help="configs[4]: number of independent 150-aa designs advanced together")
    ap.add_argument("--tensor-model", action="store_true", dest="tensor_model", help="time cdz_tm_inside (the paper's tensor-model recursion, f-4)")
    ap.add_argument("--gamma", type=int, default=4)
    ap.add_argument("--xi", type=int, default=2)
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.tensor_model:
        run_tensor_model(args)
    elif args.batch > 0:
        run_batch(args)
    else:
        run_cdz(args)


if __name__ == "__main__":
    main()
