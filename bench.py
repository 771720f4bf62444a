#!/usr/bin/env python
"""bench.py — fp64 Mcell-stage updates/s of the fused WENO5+HLLC(+viscous,+IBM) SSP-RK3 stage on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f64|f32] [--impl reference]

A "step" is one SSP-RK3 time step = 3 passes of the whole hot path (ghost fills, fused stage kernel,
CFL reduction) over the 4096x2048 throughput case of BASELINE.json configs[3].  Prints ONE JSON line.
N > 1 runs N independent replicas (the path does not shard: DESIGN.md section 7), one process per GPU.
`--impl reference` times the CPU oracle, as it stands, on a bounded sample of the same workload.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fp64 Mcell-stage updates/s (WENO5+HLLC RHS) and % of stage roofline on 1 B200"
UNIT = "Mcell-stage/s"
# algorithmic flops per cell-stage of the stage, tallied operation by operation in DESIGN.md section 6 (minimal-work
# algorithm: smoothness indicators shared by the two sides of a cell, one-sided HLLC; add / mul / compare = 1, FMA = 2,
# division = 1, square root = 1): primitives 10 + WENO5 8 x 96 + HLLC 2 x 66 + viscous 2 x 32 + divergence 20 + combine 16
# + wavespeed 6 + guard 8.  SURVEY.md section 8(d) estimated 1090 (round 1 reported against that figure; the line carries
# the fraction at both).  Compulsory bytes per cell-stage: (64 + 96 + 96) / 3.
ALG_FLOP = {"ns": 1024.0, "euler": 959.0}
ALG_FLOP_SURVEY = {"ns": 1090.0, "euler": 1000.0}
ALG_BYTES = {"f64": 85.33, "f32": 42.67}
# FP64 ALU peak derived from unit counts and clocks (B200_PROFILING.md / DESIGN.md section 6):
# 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz
PEAK_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
PEAK_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum of the stage kernel, per launch, mean of the three RK stages of one
# step, from an `ncu --set full` capture (never measured inside a bench run: a number taken under a profiler is not a
# bench value).  Each entry names the profile it was read from and the commit whose kernel was captured, so that a
# reader can tell whether it still describes the kernel being timed; None = not captured for this configuration.
NCU_TRAFFIC = {
    ("f64", 4096, 2048, "ns"): {"bytes": (525.2e6 + 842.9e6 + 800.2e6) / 3, "profile": "profiles/r02_stage.md",
                                "kernel_commit": "50169b4"},
    ("f32", 4096, 2048, "ns"): {"bytes": (238.0e6 + 398.1e6 + 374.7e6) / 3, "profile": "profiles/r02_stage.md",
                                "kernel_commit": "522b275"},
}


def max_over_ranks(ms, dist, device):
    """Timing of the slowest rank (torch.distributed MAX all-reduce; identity for a single process)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(ncell, steps, world, ms_max):
    """Whole-job Mcell-stage/s of `world` replicas that each advanced ncell cells by `steps` RK3 steps."""
    return world * ncell * 3 * steps / (ms_max * 1e-3) / 1e6


class ClockSampler:
    """SM clock, power and throttle reasons of one GPU sampled DURING the timed region.

    Source: NVML in-process (the library nvidia-smi itself reads), polled every ~2 ms from a thread, so that a timed
    region of a few tens of ms still holds samples; if NVML cannot be loaded, `nvidia-smi -lms 10` as a subprocess."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    PERIOD_S = 0.002

    def __init__(self, index):
        self.rows, self.proc, self.index, self.first = [], None, index, 0
        self.source, self._stop, self.thread, self.nv, self.h = None, threading.Event(), None, None, None
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.h = self._nvml_handle(nv, index)
            self.nv, self.source = nv, "nvml"
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nv = None
        try:
            # nvidia-smi takes a few hundred ms to print its first row: launched here, before the warm-up
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "10"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi -lms 10"
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    @staticmethod
    def _nvml_handle(nv, index):
        """NVML handle of torch's device `index` (CUDA_VISIBLE_DEVICES may renumber: match by UUID)."""
        try:
            import torch
            uuid = str(torch.cuda.get_device_properties(index).uuid)
            if not uuid.startswith("GPU-"):
                uuid = "GPU-" + uuid
            return nv.nvmlDeviceGetHandleByUUID(uuid)
        except Exception:
            return nv.nvmlDeviceGetHandleByIndex(index)

    def _poll_nvml(self):
        nv, h = self.nv, self.h
        R = nv
        bits = (("hw_slowdown", getattr(R, "nvmlClocksEventReasonHwSlowdown", 0x8)),
                ("hw_thermal_slowdown", getattr(R, "nvmlClocksEventReasonHwThermalSlowdown", 0x40)),
                ("sw_thermal_slowdown", getattr(R, "nvmlClocksEventReasonSwThermalSlowdown", 0x20)),
                ("sw_power_cap", getattr(R, "nvmlClocksEventReasonSwPowerCap", 0x4)))
        reasons_fn = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self._stop.is_set():
            try:
                mhz = float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                mask = int(reasons_fn(h))
                watts = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
                self.rows.append((mhz, self.max_mhz, watts, tuple(n for n, b in bits if mask & b)))
            except Exception:
                pass
            time.sleep(self.PERIOD_S)

    def start(self):
        t0 = time.time()
        while (self.proc or self.nv) and not self.rows and time.time() - t0 < 3.0:
            time.sleep(0.005)
        self.first = len(self.rows)

    def _read(self):
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.proc.stdout:
            f = [x.strip() for x in line.strip().split(",")]
            if len(f) < 7:
                continue
            try:
                self.rows.append((float(f[0]), float(f[1]), float(f[2]),
                                  tuple(n for n, v in zip(names, f[3:7]) if v.lower().startswith("active"))))
            except ValueError:
                continue

    def stop(self):
        if not self.proc and not self.nv:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": ["nvml and nvidia-smi unavailable"]}
        n_end = len(self.rows)
        self._stop.set()
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
        rows = self.rows[self.first:n_end]
        sm = sorted(r[0] for r in rows)
        reasons = sorted({n for r in rows for n in r[3]})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max((r[1] for r in rows), default=None),
                "sm_min_mhz": sm[0] if sm else None, "power_w_max": max((r[2] for r in rows), default=None),
                "samples": len(sm), "reasons": reasons, "source": self.source}


MIN_REGION_S = 0.25   # a timed region shorter than this is repeated back to back (see repeats_for)


def repeats_for(ms_one_call):
    """How many back-to-back repetitions of the K-step call make the timed region span MIN_REGION_S, so that the clock
    sampler sees the region (a 20-step region lasts 26 ms); the mean over the repetitions is reported."""
    return max(1, int(math.ceil(MIN_REGION_S * 1e3 / max(ms_one_call, 1e-3))))


def oracle_rate(case, nsteps):
    """Mcell-stage/s of the CPU oracle (single thread) on `case` for nsteps RK3 steps."""
    from oracle import jxo
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"])
    if case.get("phi") is not None:
        o.set_ibm(case["phi"])
    t0 = time.perf_counter()
    o.step(case["U0"], 0.4, nsteps)
    dt = time.perf_counter() - t0
    return case["nx"] * case["ny"] * 3 * nsteps / dt / 1e6, dt


def oracle_rate_1d(kind, skip):
    """cpu_baseline of the one-dimensional workloads: the oracle (one thread) on a bounded sample of the same tube,
    as the planar problem of 8 identical rows it uses everywhere for 1D (so 8 nx cells are computed per stage).
    kind: 'step' | 'tangent' | 'adjoint' (= one tangent run per entry of the state: the transpose from its definition)."""
    if skip:
        return None
    import numpy as np
    from oracle import jxo
    from paper_2601_04400_b200 import workloads as wl
    nx, ns = {"step": (40000, 20), "tangent": (20000, 15), "adjoint": (128, 6)}[kind]  # about 10 s each
    c1 = wl.sod1d(nx, gamma=1.3)
    c = wl.as_rows(c1)
    o = jxo.Oracle(c["nx"], c["ny"], c["dx"], c["dy"], c["gamma"], c["mu"], c["Pr"], c["bc"])
    dt = 0.2 * c["dx"]
    t0 = time.perf_counter()
    if kind == "step":
        o.step_fixed_dt(c["U0"], dt, ns)
    elif kind == "tangent":
        o.step_fixed_dt_tangent(c["U0"], np.repeat(wl.dcons_dgamma(c1["U0"], 1.3), 8, axis=1), 1.0, dt, ns)
    else:
        o.step_fixed_dt_adjoint(c["U0"], np.ones((4, 1, nx)), dt, ns, planar=True)
    el = time.perf_counter() - t0
    return {"value": nx * 3 * ns / el / 1e6, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"1D Sod tube at {nx} cells (as 8 identical rows: 8 x {nx} cells computed), {ns} RK3 steps, "
                      f"{kind}, {el:.1f} s, 1 thread"}


def run_reference(args, rank):
    """The reference arm = the oracle on the host cores; rank 0 only."""
    if rank != 0:
        return
    from paper_2601_04400_b200 import workloads as wl
    from oracle import jxo
    nx, ny = 512, 256
    case = wl.throughput_case(nx, ny)
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"])
    o.set_ibm(case["phi"])
    U = case["U0"]
    for _ in range(args.warmup):
        U = o.step(U, 0.4, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        U = o.step(U, 0.4, 1)
    dt = time.perf_counter() - t0
    val = nx * ny * 3 * args.steps / dt / 1e6
    sample = (f"throughput case (8 seeded cylinders, Mach 3, Re 1e5, IBM) generated at {nx}x{ny} instead of 4096x2048; "
              f"{args.steps} RK3 steps per run, 1 thread")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "throughput_4096x2048 (BASELINE.json configs[3]) sampled at 512x256", "cfl": 0.4},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_sod1d(args, rank, world, local_rank, dist, barrier, tdt):
    """the paper's 1D Sod workload at 9e6 degrees of freedom (3e6 cells x 3
    variables) through the one-dimensional stage kernel, SSP-RK3 with the CFL step on the device."""
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl
    nx = 3_000_000
    case = wl.sod1d(nx)
    stream = torch.cuda.current_stream()
    solver = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    U = torch.tensor(case["U0"], dtype=tdt, device="cuda")
    K, W = args.steps, args.warmup
    sampler = ClockSampler(local_rank)
    solver.step(U, 0.4, W)
    solver.set_profiling(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    e0.record(stream)
    solver.step(U, 0.4, K)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    stage_ms, stage_n = solver.stage_time()
    if not bool(torch.isfinite(U).all()):
        raise SystemExit("bench.py: non-finite state after the timed region")
    if rank != 0:
        return
    # one-dimensional stage: WENO 4 x 97 + HLLC 85 + primitives 10 + divergence 8 + RK 16 + wavespeed 8 flop, 85.33 B
    flop = 515.0
    avg = stage_ms / max(stage_n, 1)
    achieved = flop * nx / (avg * 1e-3) / 1e12
    peak = PEAK_FP64_TFLOPS if args.dtype == "f64" else PEAK_FP32_TFLOPS
    print(json.dumps({
        "metric": METRIC, "value": aggregate_rate(nx, K, world, ms), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": "sod1d_3000000 (the paper's 1D Sod tube at 9e6 degrees of freedom, PAPER.md L149)", "cfl": 0.4,
                   "rk": "SSP-RK3", "cells": nx, "l2": "3 x 96 MB of state buffers vs 126 MB of L2, no flush needed",
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": solver.launch_count() - launches0,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                     "traffic": None, "kernel": "jxs::stage1d_kernel", "avg_launch_ms": avg, "launches_timed": stage_n,
                     "alg_flop_per_cell_stage": flop, "alg_bytes_per_cell_stage": ALG_BYTES[args.dtype],
                     "hbm_side_gbs": ALG_BYTES[args.dtype] * nx / (avg * 1e-3) / 1e9},
        "e2e": None, "cpu_baseline": oracle_rate_1d("step", args.no_cpu_baseline)}))


def run_tangent1d(args, rank, world, local_rank, dist, barrier, tdt):
    """SURVEY.md section 8(f) rank 3 (forward mode): the 1D Sod tube at 3e6 cells stepped together with its tangent
    with respect to gamma (Eq. 16), then the loss of Eq. 14 and dL/dgamma: one iteration of the gamma
    inference per call."""
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl
    if args.dtype != "f64":
        raise SystemExit("bench.py: the tangent is fp64 only")
    nx = 3_000_000
    case = wl.sod1d(nx, gamma=1.3)
    dt = 0.2 * case["dx"]
    stream = torch.cuda.current_stream()
    solver = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    U = torch.tensor(case["U0"], dtype=tdt, device="cuda")
    D = torch.tensor(wl.dcons_dgamma(case["U0"], case["gamma"]), dtype=tdt, device="cuda")
    target = torch.tensor(wl.sod1d(nx)["U0"], dtype=tdt, device="cuda")
    K, W = args.steps, args.warmup
    solver.step_fixed_dt_tangent(U, D, 1.0, dt, W)
    solver.set_profiling(True)
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    e0.record(stream)
    solver.step_fixed_dt_tangent(U, D, 1.0, dt, K)
    loss, dloss = solver.mse_tangent(U, D, target)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    stage_ms, stage_n = solver.stage_time()
    if not (bool(torch.isfinite(U).all()) and bool(torch.isfinite(D).all()) and math.isfinite(dloss)):
        raise SystemExit("bench.py: non-finite state or tangent after the timed region")
    if rank != 0:
        return
    # value + derivative of the 1D Euler stage, counted operation by operation in DESIGN.md section 6: 1201 flop and
    # (128 + 192 + 192) / 3 B per cell-stage
    flop, nbytes = 1201.0, 512.0 / 3.0
    avg = stage_ms / max(stage_n, 1)
    achieved = flop * nx / (avg * 1e-3) / 1e12
    print(json.dumps({
        "metric": METRIC, "value": aggregate_rate(nx, K, world, ms), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": "tangent1d_3000000 (1D Sod tube stepped with its tangent with respect to gamma, then the "
                               "loss of Eq. 14 and dL/dgamma; PAPER.md Eq. 16, L149)", "dt": dt, "rk": "SSP-RK3",
                   "cells": nx, "l2": "6 x 96 MB of state and tangent buffers vs 126 MB of L2, no flush needed",
                   "loss": loss, "dloss_dgamma": dloss, "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": solver.launch_count() - launches0,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": PEAK_FP64_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / PEAK_FP64_TFLOPS, "traffic": None, "kernel": "jxs::tangent1d_kernel",
                     "avg_launch_ms": avg, "launches_timed": stage_n, "alg_flop_per_cell_stage": flop,
                     "alg_bytes_per_cell_stage": nbytes, "hbm_side_gbs": nbytes * nx / (avg * 1e-3) / 1e9},
        "e2e": None, "cpu_baseline": oracle_rate_1d("tangent", args.no_cpu_baseline)}))


def run_adjoint1d(args, rank, world, local_rank, dist, barrier, tdt):
    """SURVEY.md section 8(f) rank 3 (reverse mode): one iteration of the gamma inference by backpropagation
     on the 1D Sod tube at 3e6 cells: K recorded steps, dL/dU of Eq. 14, K adjoint steps."""
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl
    if args.dtype != "f64":
        raise SystemExit("bench.py: the adjoint is fp64 only")
    nx = 3_000_000
    case = wl.sod1d(nx, gamma=1.3)
    dt = 0.2 * case["dx"]
    stream = torch.cuda.current_stream()
    solver = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    U0 = torch.tensor(case["U0"], dtype=tdt, device="cuda")
    seed = torch.tensor(wl.dcons_dgamma(case["U0"], case["gamma"]), dtype=tdt, device="cuda")
    target = torch.tensor(wl.sod1d(nx)["U0"], dtype=tdt, device="cuda")
    K, W = args.steps, args.warmup

    def iteration(n):
        U = U0.clone()
        solver.step_fixed_dt_record(U, dt, n)
        B = (U - target).mul_(2.0 / U.numel())         # dL/dU of Eq. 14
        gbar = solver.adjoint_steps(B)
        return gbar + float((B * seed).sum())           # dL/dgamma at fixed primitives (R23)

    iteration(W)
    # untimed: the first call sizes the handle's tape for K steps (one allocation, kept between calls) and runs as plain
    # launches, the second captures the forward and the reverse sweep as CUDA graphs, the third replays them
    for _ in range(3):
        iteration(K)
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    e0.record(stream)
    dloss = iteration(K)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    launches1 = solver.launch_count()
    solver.set_profiling(True)                         # plain launches with events around the adjoint kernel: the roofline
    iteration(K)
    solver.set_profiling(False)
    stage_ms, stage_n = solver.stage_time()            # the adjoint kernel's launches of the reverse sweep
    if not math.isfinite(dloss):
        raise SystemExit("bench.py: non-finite gradient after the timed region")
    if rank != 0:
        return
    # adjoint of the 1D Euler stage: the stage's values recomputed (471 flop) + the reverse sweep (581) + the combine
    # (16); bytes: state, adjoint in, adjoint out (+ two more adjoints in the first stage)
    flop, nbytes = 1068.0, (96.0 + 96.0 + 160.0) / 3.0
    avg = stage_ms / max(stage_n, 1)
    achieved = flop * nx / (avg * 1e-3) / 1e12
    print(json.dumps({
        "metric": METRIC, "value": aggregate_rate(nx, K, world, ms), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": "adjoint1d_3000000 (1D Sod tube: K recorded steps, dL/dU of Eq. 14, K adjoint steps; one "
                               "cell-stage = forward + reverse; PAPER.md L115-128, L149)", "dt": dt, "rk": "SSP-RK3",
                   "cells": nx, "l2": "the recorded trajectory (288 MB per step) streams through HBM, no flush needed",
                   "dloss_dgamma": dloss, "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": launches1 - launches0,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": PEAK_FP64_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / PEAK_FP64_TFLOPS, "traffic": None, "kernel": "jxs::adjoint1d_kernel",
                     "avg_launch_ms": avg, "launches_timed": stage_n, "alg_flop_per_cell_stage": flop,
                     "alg_bytes_per_cell_stage": nbytes, "hbm_side_gbs": nbytes * nx / (avg * 1e-3) / 1e9},
        "e2e": None, "cpu_baseline": oracle_rate_1d("adjoint", args.no_cpu_baseline)}))


def run_adjoint2d(args, rank, world, local_rank, dist, barrier, tdt):
    """SURVEY.md section 8(f) rank 3 in two dimensions: one iteration of the gamma inference by backpropagation on the
    shock-cylinder case of BASELINE.json configs[2] (1024 x 512, Navier-Stokes, IBM; Fig. 5d-f): K recorded
    steps, dL/dU of Eq. 14, K adjoint steps through deriv2d_kernels.cuh."""
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl
    if args.dtype != "f64":
        raise SystemExit("bench.py: the adjoint is fp64 only")
    nx, ny = 1024, 512
    case = wl.shock_cylinder(nx, ny, Ms=2.0, gamma=1.35, x_shock=0.29)
    ncell = nx * ny
    stream = torch.cuda.current_stream()
    solver = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    U0 = torch.tensor(case["U0"], dtype=tdt, device="cuda")
    solver.step(U0, 0.4, 40)                      # the shock is on the body
    dt = solver.time()[1]
    seed = torch.tensor(wl.dcons_dgamma(U0.cpu().numpy(), case["gamma"]), dtype=tdt, device="cuda")
    target = U0 * 1.001
    K, W = args.steps, args.warmup

    def iteration(n):
        U = U0.clone()
        solver.step_fixed_dt_record(U, dt, n)
        B = (U - target).mul_(2.0 / U.numel())
        gbar = solver.adjoint_steps(B)
        return gbar + float((B * seed).sum())

    iteration(W)
    for _ in range(3):   # plain launches, capture of the two sweeps as CUDA graphs, replay
        iteration(K)
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    e0.record(stream)
    dloss = iteration(K)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    launches1 = solver.launch_count()
    solver.set_profiling(True)                    # plain launches with events around the adjoint stages: the roofline
    iteration(K)
    solver.set_profiling(False)
    stage_ms, stage_n = solver.stage_time()       # per adjoint stage: the two line passes, transposes, viscous kernels
    if not math.isfinite(dloss):
        raise SystemExit("bench.py: non-finite gradient after the timed region")
    if rank != 0:
        return
    # per cell and adjoint stage: each of the two line passes recomputes the direction's values
    # (471 flop) and reverses them (581); the viscous operator forward (65) and reversed (130); the combine 16
    flop = 2 * (471.0 + 581.0) + 65.0 + 130.0 + 16.0
    avg = stage_ms / max(stage_n, 1)
    achieved = flop * ncell / (avg * 1e-3) / 1e12
    print(json.dumps({
        "metric": METRIC, "value": aggregate_rate(ncell, K, world, ms), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": "adjoint2d_1024x512 (shock-cylinder case of configs[2]: K recorded steps, dL/dU of Eq. 14, K "
                               "adjoint steps; one cell-stage = forward + reverse; PAPER.md L115-128, L170)", "dt": dt,
                   "rk": "SSP-RK3", "cells": ncell, "l2": "the recorded trajectory (51 MB per step) and the transposed "
                   "scratch fields stream through L2 / HBM", "dloss_dgamma": dloss,
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": launches1 - launches0,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": PEAK_FP64_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / PEAK_FP64_TFLOPS, "traffic": None,
                     "kernel": "one adjoint stage = 2 x jxs::adjoint_line_kernel + 3 x transpose_swap_kernel + 3 viscous2d_adjoint kernels",
                     "avg_launch_ms": avg, "launches_timed": stage_n, "alg_flop_per_cell_stage": flop},
        "e2e": None, "cpu_baseline": None}))


def run_train1d(args, rank, world, local_rank, dist, barrier, tdt):
    """SURVEY.md section 8(f) rank 3, the paper's second mode (Fig. 3c): one training iteration
    of the 1D neural flux at the paper's low resolution N = 500 — K unrolled steps recorded with the per-face MLP in
    every stage, then the reverse sweep driven by Eq. 14 with one block-averaged N = 1000 target per unrolled step
    (jxs_adjoint_steps_mse) through solver and network, the weights' gradient copied out."""
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl
    if args.dtype != "f64":
        raise SystemExit("bench.py: the adjoint is fp64 only")
    nx = 500
    case = wl.sod1d(nx)
    dt = 0.2 * case["dx"]
    stream = torch.cuda.current_stream()
    solver = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    solver.set_flux_mlp(wl.mlp_weights(7), *wl.mlp_scales(out_factor=5e-2))
    U0 = torch.tensor(case["U0"], dtype=tdt, device="cuda")
    hi = wl.sod1d(2 * nx)
    Uh = torch.tensor(hi["U0"], dtype=tdt, device="cuda")
    K, W = args.steps, args.warmup
    fine = jxs.Solver.from_case(hi, dtype=tdt, stream=stream)
    targets = torch.empty((max(K, W), 4, 1, nx), dtype=tdt, device="cuda")
    for k in range(max(K, W)):   # d(U_HR^{n+s}), s = 1 .. K: block averages of the N = 1000 run, one per unrolled step
        fine.step_fixed_dt(Uh, 0.5 * dt, 2)
        targets[k] = 0.5 * (Uh[:, :, 0::2] + Uh[:, :, 1::2])
    B = torch.empty_like(U0)

    def iteration(n):
        U = U0.clone()
        solver.step_fixed_dt_record(U, dt, n)
        solver.adjoint_steps_mse(targets[:n].contiguous(), B)     # Eq. 14 over the n unrolled steps and its gradients
        return solver.flux_mlp_gradient()

    iteration(W)
    for _ in range(3):   # plain launches, capture of the two sweeps as CUDA graphs, replay
        iteration(K)
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    e0.record(stream)
    g = iteration(K)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    launches1 = solver.launch_count()
    solver.set_profiling(True)   # plain launches with events around the adjoint kernel: the roofline's launch time
    iteration(K)
    solver.set_profiling(False)
    stage_ms, stage_n = solver.stage_time()
    if not all(map(math.isfinite, g)):
        raise SystemExit("bench.py: non-finite gradient after the timed region")
    if rank != 0:
        return
    flop = 1068.0
    avg = stage_ms / max(stage_n, 1)
    achieved = flop * nx / (avg * 1e-3) / 1e12
    print(json.dumps({
        "metric": METRIC, "value": aggregate_rate(nx, K, world, ms), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": "train1d_500 (one training iteration of the 1D neural flux at the paper's N = 500 against the "
                               "block-averaged N = 1000 run: K unrolled steps forward with the MLP, backward through solver "
                               "and network; P:L109, L112-128)", "dt": dt, "rk": "SSP-RK3", "cells": nx,
                   "l2": "everything fits in L2: the iteration is bound by its 22 launches per step, not by bandwidth",
                   "grad_norm": float(sum(x * x for x in g) ** 0.5),
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": launches1 - launches0,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": PEAK_FP64_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / PEAK_FP64_TFLOPS, "traffic": None, "kernel": "jxs::adjoint1d_kernel",
                     "avg_launch_ms": avg, "launches_timed": stage_n, "alg_flop_per_cell_stage": flop,
                     "note": "500 cells = 5 CTAs: launch latency, not arithmetic, sets these times"},
        "e2e": None, "cpu_baseline": None}))


def run_cnn(args, rank, world, local_rank, dist, barrier, tdt):
    """the C4 grid with the paper's 2D CNN neural flux (Eq. 11-13) in
    every stage: reconstruction pass + 3 convolution layers per direction on tcgen05, then the stage kernel."""
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl
    case = wl.throughput_case(args.nx, args.ny)
    ncell = args.nx * args.ny
    stream = torch.cuda.current_stream()
    solver = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    solver.set_flux_cnn(wl.cnn_weights(), *wl.cnn_scales())
    U = torch.tensor(case["U0"], dtype=tdt, device="cuda")
    K, W = args.steps, args.warmup
    sampler = ClockSampler(local_rank)
    solver.step(U, 0.4, W)
    solver.set_profiling(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = solver.launch_count()
    barrier()
    sampler.start()
    e0.record(stream)
    solver.step(U, 0.4, K)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    stage_ms, stage_n = solver.stage_time()
    net_ms, net_n = solver.flux_mlp_time()
    if not bool(torch.isfinite(U).all()):
        raise SystemExit("bench.py: non-finite state after the timed region")
    if rank != 0:
        return
    # network roofline: 2 (36*32 + 288*16 + 144*4) = 12 672 flop per face, 2 faces per cell, bf16 tensor cores
    flop = 2.0 * 12672.0 * ncell
    avg = net_ms / max(net_n, 1)
    peak = 1376.0
    try:
        peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["bf16_tflops_sustained"]
    except Exception:
        pass
    print(json.dumps({
        "metric": METRIC, "value": aggregate_rate(ncell, K, world, ms), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
        "data": "synthetic",
        "config": {"workload": f"throughput_{args.nx}x{args.ny} with the paper's 2D CNN neural flux (6388 parameters, bf16) in every stage",
                   "cfl": 0.4, "rk": "SSP-RK3", "cells": ncell, "l2": "state and activation fields far larger than L2, no flush needed",
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": solver.launch_count() - launches0,
        "roofline": {"bound": "tensor", "achieved": flop / (avg * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                     "frac": flop / (avg * 1e-3) / 1e12 / peak, "traffic": None,
                     "kernel": "jxs::cnn_recon_kernel + 2 x jxs::cnn_fused_kernel (one network pass)",
                     "avg_launch_ms": avg, "launches_timed": net_n, "stage_kernel_avg_launch_ms": stage_ms / max(stage_n, 1),
                     "alg_flop_per_cell_stage": 2.0 * 12672.0,
                     "peak_source": "MEASURED_PEAKS.json bf16_tflops_sustained (dense bf16)"},
        "e2e": None, "cpu_baseline": None}))


def run_c5(args, rank, world, local_rank, dist, barrier, tdt):
    """BASELINE.json configs[4]: 16 handles x (1024x512 shock-cylinder, Mach ~ U[1.5,3]) with the bf16 flux MLP
    fused into the fp64 HLLC flux; one stream per handle, jxs_step_async on each, aggregate Mcell-stage/s."""
    import numpy as np
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl
    cases = wl.batch_cases(16)
    w, (ins, outs) = wl.mlp_weights(), wl.mlp_scales()
    ngroups = args.batch_groups if args.batch_groups > 0 else len(cases)
    streams = [torch.cuda.Stream() for _ in range(ngroups)]
    solvers, Us = [], []
    if args.batch_groups > 0:
        # batched handles (jxs_create_batch): the 16 cases in `batch_groups` handles, one stream each — one launch per
        # kernel and stage for all members of a handle; two or more handles let the MUFU-bound network kernel of one
        # overlap the FP64-bound stage kernel of another
        per = (len(cases) + ngroups - 1) // ngroups
        for gi, st in enumerate(streams):
            grp = cases[gi * per:(gi + 1) * per]
            s = jxs.Solver.from_cases(grp, dtype=tdt, stream=st)
            s.set_flux_mlp(w, ins, outs)
            s.set_concurrent_handles(ngroups)
            solvers.append(s)
            Us.append(torch.tensor(np.stack([c["U0"] for c in grp]), dtype=tdt, device="cuda"))
    else:
        for c, st in zip(cases, streams):
            s = jxs.Solver.from_case(c, dtype=tdt, stream=st)
            s.set_flux_mlp(w, ins, outs)
            s.set_concurrent_handles(len(cases))
            solvers.append(s)
            Us.append(torch.tensor(c["U0"], dtype=tdt, device="cuda"))
    ncell = sum(c["nx"] * c["ny"] for c in cases)
    K, W = args.steps, args.warmup
    torch.cuda.synchronize()
    for s, U in zip(solvers, Us):
        s.step_async(U, 0.4, W)
    for s in solvers:
        s.wait()
    if args.profile_kernels:  # two event records per kernel launch: only on request, the host work is not free
        for s in solvers:
            s.set_profiling(True)
    sampler = ClockSampler(local_rank)
    main_stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def one_pass():   # K steps of every simulation, all streams released together and joined again
        for st in streams:
            st.wait_stream(main_stream)
        for s, U in zip(solvers, Us):
            s.step_async(U, 0.4, K)
        for st in streams:
            main_stream.wait_stream(st)

    e0.record(main_stream)
    one_pass()                    # untimed: how long one pass lasts decides the repetitions below
    e1.record(main_stream)
    for s in solvers:
        s.wait()
    R = 1 if args.profile_kernels else repeats_for(e0.elapsed_time(e1))
    launches0 = sum(s.launch_count() for s in solvers)
    barrier()
    sampler.start()
    e0.record(main_stream)
    for _ in range(R):
        one_pass()
    e1.record(main_stream)
    for s in solvers:
        s.wait()
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda") / R
    launches = (sum(s.launch_count() for s in solvers) - launches0) // R
    if not all(bool(torch.isfinite(U).all()) for U in Us):
        raise SystemExit("bench.py: non-finite state after the timed region")
    value = aggregate_rate(ncell, K, world, ms)
    stage_ms = sum(s.stage_time()[0] for s in solvers)
    stage_n = sum(s.stage_time()[1] for s in solvers)
    mlp_ms = sum(s.flux_mlp_time()[0] for s in solvers)
    mlp_n = sum(s.flux_mlp_time()[1] for s in solvers)
    if rank != 0:
        return
    # S5' roofline: 256 tanh per cell-stage on the MUFU units, 16 per clock per SM.  The 16
    # streams run concurrently, so per-kernel event spans overlap; the fraction is taken over the whole timed region.
    tanh_total = 256.0 * ncell * 3 * K
    mufu_peak = 148 * 16 * 1.965e9
    tanh_meas = jxs.measure_unit_rate(jxs.RATE_TANH, 100.0) * 1e12   # MUFU.TANH results per second, measured live
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": "batch_16x1024x512_flux_mlp (BASELINE.json configs[4]: 16 independent shock-cylinder runs, "
                               "Mach ~ U[1.5,3], per-face MLP 24-64-64-4 in bf16 fused into the HLLC flux)",
                   "cfl": 0.4, "rk": "SSP-RK3", "cells": ncell, "handles": len(solvers), "streams": len(streams),
                   "batched": args.batch_groups > 0,
                   "timed_region": f"{R} back-to-back passes of {K} steps of all the simulations (>= {MIN_REGION_S} s in all); "
                                   "ms_per_step and value are the mean pass",
                   "repeats": R,
                   "l2": "16 x 3 x 17 MB of state buffers = 800 MB vs 126 MB of L2, no flush needed",
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": launches,
        "roofline": {"bound": "alu", "kernel": "jxs::flux_mlp_kernel (MUFU tanh) over the whole timed region",
                     "unit": "Gtanh/s", "achieved": tanh_total / (ms * 1e-3) / 1e9, "peak": mufu_peak / 1e9,
                     "frac": tanh_total / (ms * 1e-3) / mufu_peak, "traffic": None,
                     "kernel_event_spans_ms": {"flux_mlp_kernel": mlp_ms / max(mlp_n, 1), "stage_kernel": stage_ms / max(stage_n, 1),
                                               "note": "spans on 16 concurrent streams overlap each other"},
                     "launches_timed": mlp_n,
                     "peak_source": "derived: 148 SMs x 16 MUFU/clk x 1.965 GHz (DESIGN.md section 6)",
                     "peak_measured_gtanh": tanh_meas / 1e9,
                     "frac_of_measured_tanh_rate": tanh_total / (ms * 1e-3) / tanh_meas},
        "e2e": None, "cpu_baseline": None,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--dtype", choices=("f64", "f32"), default="f64")
    ap.add_argument("--impl", choices=("jxs", "reference"), default="jxs")
    ap.add_argument("--nx", type=int, default=4096)
    ap.add_argument("--ny", type=int, default=2048)
    ap.add_argument("--euler", action="store_true", help="mu = 0, no IBM (not the headline config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--profile-kernels", action="store_true", help="c5 only: per-kernel CUDA-event spans")
    ap.add_argument("--batch-groups", type=int, default=2,
                    help="c5 only: G > 0 = the 16 cases in G batched handles (jxs_create_batch), one stream each (default 2, "
                         "the fastest measured); 0 = 16 single handles on 16 streams")
    ap.add_argument("--rows-per-segment", type=int, default=0,
                    help="fix the stage kernel's row-segment length (jxs_set_rows_per_segment) instead of measuring it at the "
                         "first step call: used for ncu captures, which would otherwise land in the ~40 tuning launches")
    ap.add_argument("--workload", choices=("c4", "c5", "sod1d", "cnn", "tangent1d", "adjoint1d", "adjoint2d", "train1d"), default="c4",
                    help="c4 = the headline throughput case (default); c5 = BASELINE.json configs[4]: 16 independent "
                         "1024x512 shock-cylinder runs with the per-face flux MLP, one stream per handle; sod1d = the "
                         "paper's 1D Sod tube at its largest size (3e6 cells = 9e6 degrees of freedom, PAPER.md L149)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "jxs" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import numpy as np
    import torch
    from paper_2601_04400_b200 import jxs, workloads as wl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the jxs path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    tdt = torch.float64 if args.dtype == "f64" else torch.float32
    if args.workload == "c5":
        run_c5(args, rank, world, local_rank, dist, barrier, tdt)
        return
    if args.workload == "sod1d":
        run_sod1d(args, rank, world, local_rank, dist, barrier, tdt)
        return
    if args.workload == "train1d":
        run_train1d(args, rank, world, local_rank, dist, barrier, tdt)
        return
    if args.workload == "adjoint1d":
        run_adjoint1d(args, rank, world, local_rank, dist, barrier, tdt)
        return
    if args.workload == "adjoint2d":
        run_adjoint2d(args, rank, world, local_rank, dist, barrier, tdt)
        return
    if args.workload == "tangent1d":
        run_tangent1d(args, rank, world, local_rank, dist, barrier, tdt)
        return
    if args.workload == "cnn":
        run_cnn(args, rank, world, local_rank, dist, barrier, tdt)
        return
    sampler = ClockSampler(local_rank)
    case = wl.throughput_case(args.nx, args.ny, viscous=not args.euler, ibm=not args.euler)
    ncell = args.nx * args.ny
    stream = torch.cuda.current_stream()
    solver = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    if args.rows_per_segment > 0:
        solver.set_rows_per_segment(args.rows_per_segment)
    U = torch.tensor(case["U0"], dtype=tdt, device="cuda")
    K, W = args.steps, args.warmup

    peak_meas = jxs.measure_fp64_peak(200.0) if args.dtype == "f64" else None
    # the same loop with three distinct vector-register operands per DFMA (x = p * q + x): 3 pipe cycles instead of 2
    peak3_meas = jxs.measure_unit_rate(jxs.RATE_DFMA3, 100.0) if args.dtype == "f64" else None

    # ---- device-resident timing: inputs already in HBM
    solver.step(U, 0.4, W)            # warm-up; the first call also measures the row-segment length (jxs_tune)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    solver.step(U, 0.4, K)            # untimed: how long one K-step call lasts decides the repetitions below
    e1.record(stream)
    torch.cuda.synchronize()
    R = repeats_for(max_over_ranks(e0.elapsed_time(e1), dist, "cuda"))
    solver.set_profiling(True)
    launches0 = solver.launch_count()
    stage_ms, stage_n = 0.0, 0
    barrier()
    sampler.start()
    e0.record(stream)
    for _ in range(R):                # R back-to-back calls of EXACTLY K steps each; the mean call is reported
        solver.step(U, 0.4, K)
        m, n = solver.stage_time()
        stage_ms, stage_n = stage_ms + m, stage_n + n
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = (solver.launch_count() - launches0) // R
    ms = e0.elapsed_time(e1) / R
    stage_ms, stage_n = stage_ms / R, stage_n // R
    solver.set_profiling(False)
    if not bool(torch.isfinite(U).all()):
        raise SystemExit("bench.py: non-finite state after the timed region")
    ms_max = max_over_ranks(ms, dist, "cuda")
    value = aggregate_rate(ncell, K, world, ms_max)

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region)
    Uh = torch.tensor(case["U0"], dtype=tdt).pin_memory()
    solver2 = jxs.Solver.from_case(case, dtype=tdt, stream=stream)
    if args.rows_per_segment > 0:
        solver2.set_rows_per_segment(args.rows_per_segment)
    solver2.step_host(Uh.clone().pin_memory(), 0.4, 3)
    barrier()
    e0.record(stream)
    for _ in range(R):
        solver2.step_host(Uh, 0.4, K)
    e1.record(stream)
    barrier()
    e2e_value = aggregate_rate(ncell, K, world, max_over_ranks(e0.elapsed_time(e1) / R, dist, "cuda"))
    nbytes = Uh.numel() * Uh.element_size()
    # the same call made once per step: the whole state crosses PCIe in both directions every step
    Kc = min(K, 10)
    barrier()
    e0.record(stream)
    for _ in range(Kc):
        solver2.step_host(Uh, 0.4, 1)
    e1.record(stream)
    barrier()
    e2e_copy_value = aggregate_rate(ncell, Kc, world, max_over_ranks(e0.elapsed_time(e1), dist, "cuda"))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the fused stage kernel): ALU-bound
    kind = "euler" if args.euler else "ns"
    stage_avg_ms = stage_ms / max(stage_n, 1)
    flops_per_launch = ALG_FLOP[kind] * ncell
    achieved = flops_per_launch / (stage_avg_ms * 1e-3) / 1e12
    peak = PEAK_FP64_TFLOPS if args.dtype == "f64" else PEAK_FP32_TFLOPS
    hbm_gbs = None
    try:
        hbm_gbs = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        pass
    traffic_rec = NCU_TRAFFIC.get((args.dtype, args.nx, args.ny, kind))
    traffic = traffic_rec["bytes"] if traffic_rec else None
    roofline = {
        "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
        "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
        "traffic_source": ({"profile": traffic_rec["profile"], "kernel_commit": traffic_rec["kernel_commit"]}
                           if traffic_rec else None),
        "kernel": "jxs::stage_kernel", "avg_launch_ms": stage_avg_ms, "launches_timed": stage_n,
        "share_of_step": stage_ms / ms,
        "alg_flop_per_cell_stage": ALG_FLOP[kind], "alg_bytes_per_cell_stage": ALG_BYTES[args.dtype],
        "alg_flop_source": "operation tally of DESIGN.md section 6",
        "frac_at_survey_estimate": ALG_FLOP_SURVEY[kind] / ALG_FLOP[kind] * achieved / peak,
        "peak_source": "derived: 148 SMs x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md section 6)",
        "peak_measured_dfma_tflops": peak_meas,
        "frac_of_measured_dfma": (achieved / peak_meas) if peak_meas else None,
        "measured_dfma_3_register_operands_tflops": peak3_meas,
        "hbm_side": {"achieved_gbs": ALG_BYTES[args.dtype] * ncell / (stage_avg_ms * 1e-3) / 1e9,
                     "peak_gbs": hbm_gbs, "peak_source": "MEASURED_PEAKS.json hbm_gbs" if hbm_gbs else None},
    }

    cpu = None
    if not args.no_cpu_baseline:
        sample_case = wl.throughput_case(1024, 512, viscous=not args.euler, ibm=not args.euler)
        ORACLE_STEPS = 24   # about 11 s of single-thread work on this box's host
        v, secs = oracle_rate(sample_case, ORACLE_STEPS)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"the same workload generated at 1024x512, {ORACLE_STEPS} RK3 steps ({3 * ORACLE_STEPS} stages), {secs:.1f} s, 1 thread"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": f"throughput_{args.nx}x{args.ny}" + ("_euler" if args.euler else
                   " (BASELINE.json configs[3]: Mach-3 shock over 8 seeded cylinders, Navier-Stokes Re 1e5, IBM)"),
                   "cfl": 0.4, "rk": "SSP-RK3", "cells": ncell, "stages_per_step": 3,
                   "timed_region": f"{R} back-to-back jxs_step calls of {K} steps each (>= {MIN_REGION_S} s in all, so that "
                                   f"the clock sampler sees the region); ms_per_step, value and e2e are the mean call",
                   "repeats": R,
                   "l2": "inputs larger than L2 (3 x 256 MiB state buffers vs 126 MB), no flush needed",
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes / K, "d2h_bytes_per_step": nbytes / K,
                "note": f"jxs_step_host calls of {K} steps on a pinned host buffer ({R} back to back, mean); bytes are one "
                        f"call's copies / {K}",
                "copies_every_step": {"value": e2e_copy_value, "unit": UNIT, "steps": Kc, "h2d_bytes_per_step": nbytes,
                                      "d2h_bytes_per_step": nbytes,
                                      "note": "jxs_step_host(nsteps = 1) per step: PCIe-bound, the state is 256 MiB"}},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
