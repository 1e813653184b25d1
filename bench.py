#!/usr/bin/env python
"""bench.py - cells*solver-iterations/s of the npFEM step on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--cells M] [--iterations I]
  python bench.py --impl reference ...        # times the fp64 CPU oracle on a bounded sample

One "step" = one npfem_step (prologue, I x (local step, global step), epilogue) over the whole
synthetic population.  Default workload: BASELINE.json configs[3], 100,000 mixed cells (90,000
RBC-642 + 10,000 PLT-162), 10 iterations per step, fp32 - the configuration the north star
quotes its target on; it fits one GPU.  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cells*solver-iterations/sec"
UNIT = "cell-iterations/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--cells", type=int, default=None, help="shrink the config to this many cells")
    ap.add_argument("--iterations", type=int, default=None, help="solver iterations per step")
    ap.add_argument("--precision", default="fp32", choices=["fp32", "fp64"])
    ap.add_argument("--global-math", default="tf32", choices=["tf32", "fp32", "tf32x2"])
    ap.add_argument("--local-impl", type=int, default=0, choices=[0, 1, 2, 3, 4, 5, 6])
    ap.add_argument("--line-search", type=int, default=0, help="Armijo backtracking with this many halvings (0 = off)")
    ap.add_argument("--graph", action="store_true",
                    help="capture one npfem_step in a CUDA graph and time replays of it (pays off at small cell counts)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-chunks", type=int, default=0, help="npfem_step_host chunks (0 = library's choice, 1 = unpipelined)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--peaks", action="store_true",
                    help="measure the FP32 FFMA, FP64 DFMA, TF32 / FP64 / BF16 GEMM and copy peaks of this box and print them "
                         "as one JSON line (kept as profiles/r2_measured_peaks.json: the roofline denominators)")
    return ap.parse_args()


NCU_RAW = {   # kernel of the bench line -> committed raw export of ONE launch of it on the bench workload
    "local:RBC-642": "r2_ncu_local_quad_rbc642_raw.csv",     # the default (quad) kernel; r2_ncu_local_sched_* = --local-impl 3
    "global:RBC-642": "r2_ncu_global_tcgen05_rbc642_raw.csv",
}
NCU_WORKLOAD = {"cells": 100000, "precision": "fp32"}   # what the exports were captured on (profiles/r2_ncu.md)


def load_ncu_raw(kernel: str):
    """Per-launch counters of a hot kernel, parsed from the committed `ncu -i <rep> --page raw --csv --print-units base`
    export of one launch (profiles/r2_ncu.md names the full commands): bench.py cannot run ncu, but every number it
    quotes from a capture is re-derivable from a tracked file.  Only valid for the workload of the capture."""
    import csv
    name = NCU_RAW.get(kernel)
    path = os.path.join(ROOT, "profiles", name) if name else None
    if not path or not os.path.exists(path):
        return None
    rows = list(csv.reader(open(path)))
    hdr, vals = rows[0], rows[2]

    def col(metric):
        for i, h in enumerate(hdr):
            if h == metric:
                return float(vals[i]) if vals[i] not in ("", "no data") else None
        return None
    # `--set full` keeps the fp32 op counts as chip-wide per-cycle sums: thread instructions = that x the elapsed cycles
    cycles = col("smsp__cycles_elapsed.avg")
    fadd, fmul, ffma = (col(f"smsp__sass_thread_inst_executed_op_{op}_pred_on.sum.per_cycle_elapsed") for op in ("fadd", "fmul", "ffma"))
    if None not in (cycles, fadd, fmul, ffma):
        fadd, fmul, ffma = fadd * cycles, fmul * cycles, ffma * cycles
    out = {"file": "profiles/" + name,
           "dram_bytes": (col("dram__bytes_read.sum") or 0) + (col("dram__bytes_write.sum") or 0),
           "warp_instructions": col("smsp__inst_executed.sum"),
           "smem_wavefronts": col("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"),
           "duration_ns_under_ncu": col("gpu__time_duration.sum"),
           "tensor_pipe_active_pct": col("sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed")}
    if None not in (fadd, fmul, ffma):
        out["fp32_flop"] = fadd + fmul + 2 * ffma
    return out


def load_peaks():
    """Measured roofline denominators: HBM and bf16 from the driver-written MEASURED_PEAKS.json (else the profiling
    guide's fallback); TF32 / FP64 GEMM and FP32 FFMA from profiles/r2_measured_peaks.json (`bench.py --peaks` on a
    B200 of this pool), else the nominal ratios, saying which."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        out = {"hbm_gbs": float(p["hbm_gbs"]), "bf16_tflops": float(p["bf16_tflops"]),
               "bf16_tflops_sustained": float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
               "sm_max_mhz": float(p.get("sm_max_mhz", 1965.0)), "source": "measured"}
    else:
        out = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
               "source": "fallback"}
    own = os.path.join(ROOT, "profiles", "r2_measured_peaks.json")
    if os.path.exists(own):
        q = json.load(open(own))
        out.update({"tf32_tflops": q["tf32_gemm_tflops"], "tf32_tflops_sustained": q["tf32_gemm_tflops_sustained"],
                    "fp64_tflops": q["fp64_gemm_tflops"], "fp32_ffma_tflops": q["fp32_ffma_tflops"],
                    "fp64_dfma_tflops": q["fp64_dfma_tflops"],
                    "own_source": "measured (profiles/r2_measured_peaks.json, bench.py --peaks)"})
    else:
        out.update({"tf32_tflops": 0.5 * out["bf16_tflops"], "tf32_tflops_sustained": 0.5 * out["bf16_tflops_sustained"],
                    "fp64_tflops": 40.0, "fp32_ffma_tflops": 148 * 128 * 2 * out["sm_max_mhz"] * 1e6 / 1e12,
                    "fp64_dfma_tflops": 40.0, "own_source": "nominal ratios (no profiles/r2_measured_peaks.json)"})
    return out


def run_peaks():
    """`--peaks`: the roofs this repository's kernels are measured against, taken on the box at hand the way
    MEASURED_PEAKS.json was (torch.matmul / copy, best of 10 and a 2 s back-to-back loop), plus the plain-ALU roofs
    from the library's own FMA probe kernel (npfem_probe_fma_peak).  Prints one JSON line."""
    import ctypes as C
    import torch
    from paper_1911_03062_b200 import binding
    lib = binding.load_library()
    torch.cuda.set_device(0)
    dev = "cuda:0"
    stream = torch.cuda.current_stream(0)

    def timed(fn, reps=10):
        fn()
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1) * 1e-3)
        return best

    def sustained(fn, seconds=2.0):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0, n = time.perf_counter(), 0
        e0.record()
        while time.perf_counter() - t0 < seconds:
            for _ in range(8):
                fn()
            n += 8
            torch.cuda.synchronize()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / n

    out = {"gpu_name": torch.cuda.get_device_name(0), "when": time.strftime("%Y-%m-%dT%H:%M:%SZ", time.gmtime()),
           "how": "bench.py --peaks: torch.matmul N^3 (2 N^3 flop; tf32 = float32 inputs with allow_tf32, fp64, bf16; N = 8192, "
                  "fp64 4096), best of 10 and back to back for 2 s; b.copy_(a) over 1 Gi bf16 (read + write bytes); "
                  "npfem_probe_fma_peak (148 x 32 CTAs x 256 threads, 16 independent FMA chains per thread), best of 10"}
    with ClockSampler(0) as clocks:
        for prec, name, iters, dt in ((binding.NPFEM_F32, "fp32_ffma_tflops", 1 << 15, torch.float32),
                                      (binding.NPFEM_F64, "fp64_dfma_tflops", 1 << 10, torch.float64)):
            sink = torch.zeros(1, dtype=dt, device=dev)
            flops = C.c_double(0.0)

            def probe():
                rc = lib.npfem_probe_fma_peak(C.c_void_p(stream.cuda_stream), prec, 148 * 32, iters, C.c_void_p(sink.data_ptr()),
                                              C.byref(flops))
                assert rc == 0
            secs = timed(probe)
            out[name] = flops.value / secs / 1e12
        torch.backends.cuda.matmul.allow_tf32 = True
        for name, dt, n in (("tf32_gemm_tflops", torch.float32, 8192), ("bf16_gemm_tflops", torch.bfloat16, 8192),
                            ("fp64_gemm_tflops", torch.float64, 4096)):
            a = torch.randn(n, n, device=dev, dtype=torch.float32).to(dt)
            b = torch.randn(n, n, device=dev, dtype=torch.float32).to(dt)
            c = torch.empty(n, n, device=dev, dtype=dt)
            fn = lambda: torch.matmul(a, b, out=c)      # noqa: E731
            out[name] = 2.0 * n ** 3 / timed(fn) / 1e12
            out[name + "_sustained"] = 2.0 * n ** 3 / sustained(fn) / 1e12
            del a, b, c
        torch.backends.cuda.matmul.allow_tf32 = False
        src = torch.empty(1 << 30, dtype=torch.bfloat16, device=dev)
        dst = torch.empty_like(src)
        out["hbm_copy_gbs"] = 2.0 * src.numel() * 2 / timed(lambda: dst.copy_(src)) / 1e9
    out["clocks"] = clocks.summary()
    print(json.dumps(out), flush=True)
    return 0


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (NVML every 10 ms; falls
    back to polling nvidia-smi when the NVML binding is missing)."""

    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, device: int):
        self.device, self.rows, self._stop, self._thread = device, [], threading.Event(), None
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            self._handle = pynvml.nvmlDeviceGetHandleByIndex(device)
            self._max = float(pynvml.nvmlDeviceGetMaxClockInfo(self._handle, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nvml = None

    def _sample_nvml(self):
        nv, h = self._nvml, self._handle
        sm = float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
        watts = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
        mask = nv.nvmlDeviceGetCurrentClocksEventReasons(h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
            else nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
        bits = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
        self.rows.append([sm, self._max, watts] + [bool(mask & bits[n]) for n in self.NAMES])

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", f"--id={self.device}", f"--query-gpu={self.QUERY}",
                              "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
        if out.returncode == 0 and out.stdout.strip():
            c = [x.strip() for x in out.stdout.strip().splitlines()[0].split(",")]
            self.rows.append([float(c[0]), float(c[1]), float(c[2])] + [x.lower().startswith("active") for x in c[3:7]])

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample_nvml() if self._nvml else self._sample_smi()
            except Exception:
                pass
            self._stop.wait(0.01 if self._nvml else 0.05)

    def __enter__(self):
        self._thread = threading.Thread(target=self._run, daemon=True)
        self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        self._thread.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock sampling unavailable"]}
        sm = sorted(r[0] for r in self.rows)
        reasons = [n for i, n in enumerate(self.NAMES) if any(r[3 + i] for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.rows[0][1], "power_w_max": max(r[2] for r in self.rows),
                "samples": len(self.rows), "reasons": reasons, "source": "nvml" if self._nvml else "nvidia-smi"}


# ---- algorithmic work per cell-iteration -------------
def algorithmic_bytes(kind: str, n: int, es: int) -> int:
    """local: read x_n, d, b, write g (4 vec3 fields); global: read g, d, write d (3 fields)."""
    return {"local": 12 * n * es, "global": 9 * n * es}[kind]


def global_flops(n: int) -> int:
    return 6 * n * n          # [3 x n] . [n x n], multiply-add = 2 flops


# ---- the oracle leg (cpu_baseline and --impl reference) --------------------------------------
def blas_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        return max([int(p.get("num_threads", 1)) for p in threadpool_info()] or [1])
    except Exception:
        return 1


def oracle_sample(pop, n_sample: int):
    """First n_sample cells of the population (same type mix) as their own population."""
    return pop.subset(np.arange(min(n_sample, pop.n_cells)))


def time_oracle(sample, n_iterations: int, busy=None) -> float:
    """Seconds for ONE time step of the oracle, as it stands, on the sample.  busy (a list) receives the process CPU
    seconds spent in the timed region: CPU seconds / wall seconds = the cores the oracle actually kept busy."""
    from oracle import npfem_oracle as orc
    tds = [orc.make_type(ct, sample.dt) for ct in sample.types]     # setup, not timed (as on the GPU)
    forces = sample.forces(0)
    c0 = os.times()
    t0 = time.perf_counter()
    for t, td in enumerate(tds):
        if sample.positions[t].shape[0]:
            orc.step(sample.positions[t], sample.velocities[t], forces[t], td, n_iterations)
    wall = time.perf_counter() - t0
    c1 = os.times()
    if busy is not None:
        busy.append((c1.user - c0.user) + (c1.system - c0.system))
    return wall


def cpu_baseline(pop, n_iterations: int, target_seconds: float):
    probe = oracle_sample(pop, min(22, pop.n_cells))
    t_probe = time_oracle(probe, n_iterations)
    per_cell = max(t_probe / probe.n_cells, 1e-6)
    n_sample = int(max(probe.n_cells, min(pop.n_cells, target_seconds / per_cell, 4000)))
    sample = oracle_sample(pop, n_sample)
    busy = []
    secs = time_oracle(sample, n_iterations, busy)
    counts = [int(np.sum(sample.type_of_cell == t)) for t in range(len(pop.types))]
    desc = " + ".join(f"{c} {ct.name}" for c, ct in zip(counts, pop.types) if c)
    cores_busy = busy[0] / secs
    return {
        # cores = what the oracle actually kept busy (process CPU seconds / wall seconds, rounded up), not what the box
        # has: it is plain numpy, whose element-wise passes and scatter-adds run on one thread; only the LAPACK /
        # BLAS calls (Cholesky solve, M~ d) fan out
        "value": sample.n_cells * n_iterations / secs, "unit": UNIT, "cores": int(max(1, np.ceil(cores_busy - 0.05))),
        "cores_busy_mean": round(cores_busy, 2), "threads_available": len(os.sched_getaffinity(0)),
        "blas_threads": blas_threads(), "kind": "oracle",
        "sample": f"first {sample.n_cells} cells of the workload ({desc}), 1 step x {n_iterations} iterations, "
                  f"{secs:.1f} s wall, {busy[0]:.1f} CPU s",
    }, sample


def run_reference(args, pop, n_iterations: int, config_desc: dict):
    """--impl reference: the fp64 oracle as it stands, each step a bounded sample of the workload."""
    info, sample = cpu_baseline(pop, n_iterations, args.cpu_seconds)
    for _ in range(min(args.warmup, 1)):
        time_oracle(sample, n_iterations)
    times = [time_oracle(sample, n_iterations) for _ in range(args.steps)]
    total = float(np.sum(times))
    value = sample.n_cells * n_iterations * args.steps / total
    info["value"] = value
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_desc, "cpu_baseline": info,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


# ---- multi-rank plumbing (one process per GPU, replicas only: DESIGN.md section 8) ---------------
def max_over_ranks(value_ms: float, world: int, device: str) -> float:
    """Device time of the slowest rank (all_reduce MAX); identity for one rank."""
    if world <= 1:
        return float(value_ms)
    import torch
    t = torch.tensor([value_ms], device=device, dtype=torch.float64)
    torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(cells_per_rank: int, n_iterations: int, steps: int, world: int, max_ms: float) -> float:
    """Whole-job cells*iterations/s: every rank advances its own replica (weak scaling), the clock is
    the slowest rank's."""
    return world * cells_per_rank * n_iterations * steps / (max_ms * 1e-3)


# ---- the B200 arm ------------------------------------------------------------------------------
def run_b200(args, pop, n_iterations: int, config_desc: dict, rank: int, world: int):
    import torch
    from paper_1911_03062_b200 import Solver, binding

    local_rank = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    es = 4 if args.precision == "fp32" else 8
    np_io = np.float32 if args.precision == "fp32" else np.float64
    peaks = load_peaks()

    if args.graph:      # a graph cannot be captured on the legacy default stream: the whole run moves to a side stream
        torch.cuda.set_stream(torch.cuda.Stream(device=local_rank))
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=args.precision, device=local_rank)
    solver.set_option(binding.OPT_GLOBAL_STEP_MATH, {"tf32": 0, "fp32": 1, "tf32x2": 2}[args.global_math])
    solver.set_option(binding.OPT_LOCAL_STEP_IMPL, args.local_impl)
    if args.line_search:
        solver.set_line_search(args.line_search)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).to(dev))
    forces_host = torch.from_numpy(pop.packed(pop.forces(0), dtype=np_io)).pin_memory()
    forces_dev = forces_host.to(dev)
    solver.set_forces(forces_dev)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: inputs already in HBM -------------------------------------
    for _ in range(args.warmup):
        solver.step(n_iterations)
    barrier()
    graph, launches_per_step = None, None
    if args.graph:
        # npfem_step allocates nothing and never synchronises (include/npfem.h): one step = one capturable sequence
        l0 = solver.launch_count
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=torch.cuda.current_stream(local_rank)):
            solver.step(n_iterations)
        launches_per_step = solver.launch_count - l0
        graph.replay()
        barrier()
    launches0 = solver.launch_count
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(local_rank) as clocks:
        marks[0].record()
        for k in range(args.steps):
            if graph is not None:
                graph.replay()
            else:
                solver.step(n_iterations)
            marks[k + 1].record()                     # one event between steps: per-step times for median / best
        barrier()
    elapsed_ms = marks[0].elapsed_time(marks[-1])
    step_ms = sorted(marks[k].elapsed_time(marks[k + 1]) for k in range(args.steps))
    launches = launches_per_step * args.steps if graph is not None else solver.launch_count - launches0
    # per-kernel breakdown: the same K steps again with a CUDA-event pair around every launch (kept out of
    # the timed region above: the events cost as much as a small kernel in the small-batch regime)
    solver.set_option(binding.OPT_KERNEL_TIMING, 1)
    solver.get_kernel_times(reset=True)
    for _ in range(args.steps):
        solver.step(n_iterations)
    ktimes = solver.get_kernel_times(reset=True)
    solver.set_option(binding.OPT_KERNEL_TIMING, 0)
    elapsed_ms = max_over_ranks(elapsed_ms, world, dev)
    # the fp32 default path must have run the tcgen05 GEMM: the SIMT GEMM is a different kernel kind and never a
    # silent fallback (include/npfem.h NPFEM_KIND_GLOBAL_SIMT)
    simt_launches = sum(n for _, n in ktimes["global_simt"])
    if args.precision == "fp32" and args.global_math != "fp32" and simt_launches:
        raise RuntimeError(f"the fp32 tensor-core path launched the SIMT GEMM {simt_launches} times: refusing to report")
    cell_iters = pop.n_cells * n_iterations * args.steps
    value = aggregate_throughput(pop.n_cells, n_iterations, args.steps, world, elapsed_ms)

    # ---- per-kernel rooflines from the live CUDA-event times ---------------------------------
    kernels, total_kernel_ms = [], sum(ms for v in ktimes.values() for ms, _ in v)
    for kind in ("local", "global", "global_simt"):
        for t, ct in enumerate(pop.types):
            ms, cnt = ktimes[kind][t]
            cells_t = int(np.sum(pop.type_of_cell == t))
            if cnt == 0 or cells_t == 0:
                continue
            per_launch_s = ms * 1e-3 / cnt
            bytes_launch = algorithmic_bytes("local" if kind == "local" else "global", ct.n_vertices, es) * cells_t
            row = {"kernel": f"{kind}:{ct.name}", "launches": cnt, "avg_ms": ms / cnt,
                   "share_of_kernel_time": ms / total_kernel_ms,
                   "hbm_gbs": bytes_launch / per_launch_s / 1e9,
                   "hbm_frac": bytes_launch / per_launch_s / 1e9 / peaks["hbm_gbs"]}
            if kind != "local":
                tflops = global_flops(ct.n_vertices) * cells_t / per_launch_s / 1e12
                # TF32 / FP64 dense GEMM peaks: measured on the box by `bench.py --peaks` (profiles/r2_measured_peaks.json),
                # the sustained figure because the kernel is timed inside a long step
                row["tflops"] = tflops
                if kind == "global":
                    row["tensor_frac_tf32"] = tflops / peaks["tf32_tflops_sustained"]
                else:
                    row["frac_of_" + ("fp64_gemm" if args.precision == "fp64" else "fp32_ffma") + "_peak"] = \
                        tflops / (peaks["fp64_tflops"] if args.precision == "fp64" else peaks["fp32_ffma_tflops"])
                row["peak_source"] = peaks["own_source"]
            kernels.append(row)
    dominant = max(kernels, key=lambda r: r["share_of_kernel_time"]) if kernels else None
    roofline = None
    same_workload = NCU_WORKLOAD["cells"] == pop.n_cells and NCU_WORKLOAD["precision"] == args.precision and \
        args.global_math == "tf32" and args.local_impl == 0 and not args.line_search
    if dominant:
        cap = load_ncu_raw(dominant["kernel"]) if same_workload else None
        roofline = {"kernel": dominant["kernel"], "bound": "hbm", "achieved": dominant["hbm_gbs"],
                    "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": dominant["hbm_frac"],
                    "traffic": cap["dram_bytes"] if cap else None,
                    "traffic_source": cap["file"] if cap else None,
                    "peak_source": peaks["source"] + " (MEASURED_PEAKS.json hbm_gbs)",
                    "note": "north_star names HBM for the local step; the kernel is bound by instruction issue and "
                            "shared-memory wavefronts (DESIGN.md 7.1), see `alu`"}
        if cap and cap.get("warp_instructions"):
            # plain-ALU roofline: 148 SMs x 4 schedulers x 1 warp instruction / cycle at the max SM clock
            sm_mhz = peaks.get("sm_max_mhz", 1965.0)
            alu_peak = 148 * 4 * sm_mhz * 1e6
            ach = cap["warp_instructions"] / (dominant["avg_ms"] * 1e-3)
            roofline["alu"] = {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "warp-instructions/s",
                               "frac": ach / alu_peak, "smem_wavefronts_per_launch": cap.get("smem_wavefronts")}
            if cap.get("fp32_flop"):
                # achieved FP32 FLOP/s (fadd + fmul + 2 ffma, ncu op counts) against
                # 148 SMs x 128 lanes x 2 x the max SM clock
                fp32_peak = peaks["fp32_ffma_tflops"]
                tf = cap["fp32_flop"] / (dominant["avg_ms"] * 1e-3) / 1e12
                roofline["fp32"] = {"achieved": tf, "peak": fp32_peak, "unit": "TFLOP/s", "frac": tf / fp32_peak,
                                    "peak_source": peaks["own_source"]}
    for row in kernels:
        cap = load_ncu_raw(row["kernel"]) if same_workload else None
        row["traffic"] = cap["dram_bytes"] if cap else None
        if cap and cap.get("tensor_pipe_active_pct") is not None and row["kernel"].startswith("global"):
            row["tensor_pipe_active_pct_ncu"] = cap["tensor_pipe_active_pct"]

    result = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32" if args.precision == "fp32" else "f64",
        "data": "synthetic", "config": config_desc, "clocks": clocks.summary(), "gpu_launches": launches,
        "ms_per_step_median": step_ms[len(step_ms) // 2] if len(step_ms) % 2 else 0.5 * (step_ms[len(step_ms) // 2 - 1] + step_ms[len(step_ms) // 2]),
        "ms_per_step_best": step_ms[0],
        "roofline": roofline, "kernels": kernels,
        "kernel_ms_per_step": {k: sum(ms for ms, _ in v) / args.steps for k, v in ktimes.items()},
    }

    # ---- end to end through the C-ABI with HOST buffers ------------------------------------
    if not args.no_e2e:
        count = 3 * solver.total_vertices
        pos_host = torch.empty(count, dtype=forces_host.dtype).pin_memory()
        vel_host = torch.empty(count, dtype=forces_host.dtype).pin_memory()
        for _ in range(2):
            solver.step_host(forces_host, n_iterations, pos_host, vel_host, n_chunks=args.e2e_chunks)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            # npfem_step_host: H2D of this step's F_ext, the step, D2H of {x, v}; pipelined over chunks of
            # cells inside the call, which returns with the state in the host buffers
            solver.step_host(forces_host, n_iterations, pos_host, vel_host, n_chunks=args.e2e_chunks)
        e1.record()
        barrier()
        e2e_ms = e0.elapsed_time(e1)
        e2e_ms = max_over_ranks(e2e_ms, world, dev)
        result["e2e"] = {"value": aggregate_throughput(pop.n_cells, n_iterations, args.steps, world, e2e_ms), "unit": UNIT,
                         "h2d_bytes_per_step": int(forces_host.numel() * forces_host.element_size()),
                         "d2h_bytes_per_step": int(2 * count * pos_host.element_size()),
                         "ms_per_step": e2e_ms / args.steps,
                         "call": "npfem_step_host", "chunks": args.e2e_chunks}
    solver.close()
    return result


def main():
    args = parse_args()
    if args.peaks:
        return run_peaks()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    from workloads import CONFIG_NAMES, make_config
    n_iterations = args.iterations

    if args.impl == "reference":
        if rank != 0:
            return 0
        args.cpu_seconds = min(args.cpu_seconds, 120.0 / max(args.steps, 1))
        small = make_config(args.config, n_cells=min(args.cells or 10 ** 9, 4400))
        full_cells = args.cells or make_config_size(args.config)
        n_iterations = n_iterations or small.n_iterations
        desc = config_description(args, small, full_cells, n_iterations)
        print(json.dumps(run_reference(args, small, n_iterations, desc)), flush=True)
        return 0

    import torch
    if world > 1:
        torch.distributed.init_process_group("nccl")
    pop = make_config(args.config, n_cells=args.cells)
    n_iterations = n_iterations or pop.n_iterations
    desc = config_description(args, pop, pop.n_cells, n_iterations)
    desc["parallelism"] = f"{world} independent replica(s) of the workload, one per GPU, no collective"
    result = run_b200(args, pop, n_iterations, desc, rank, world)
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            result["cpu_baseline"], _ = cpu_baseline(pop, n_iterations, args.cpu_seconds)
        print(json.dumps(result), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


def make_config_size(index: int) -> int:
    return {1: 1, 2: 1000, 3: 22000, 4: 100000, 5: 10000, 6: 114}[index]


def config_description(args, pop, n_cells: int, n_iterations: int) -> dict:
    from workloads import CONFIG_NAMES
    mix = {ct.name: ct.n_vertices for ct in pop.types}
    label = f"BASELINE.json configs[{args.config - 1}]" if args.config <= 5 else "SURVEY.md 8(f)-3 (not a BASELINE config)"
    return {"workload": f"{label}: {CONFIG_NAMES[args.config]}",
            "cells": int(n_cells), "cell_types_vertices": mix, "iterations_per_step": int(n_iterations),
            "dt_us": pop.dt, "precision": args.precision, "global_step_math": args.global_math,
            "line_search_halvings": int(args.line_search), "cuda_graph": bool(args.graph),
            "l2": ("no flush needed: the state touched per iteration (>= 2.9 GB at 100k cells) exceeds the 126 MB L2"
                   if n_cells >= 20000 else "state fits the 126 MB L2: small-batch latency regime, no flush")}


if __name__ == "__main__":
    sys.exit(main())
