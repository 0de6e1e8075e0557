#!/usr/bin/env python
"""bench.py -- spin-updates/s of the LLG hot path on B200 (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--inner 100]

One bench "step" = one `llg_iterate(inner)` call = `inner` (default 128) Depondt iterations (each: field of every spin at n,
predictor, field at n^p, corrector; all rows of SURVEY 8(a)) over the whole lattice.  Workload at N=1: configs[2] of
BASELINE.json, the 3-D simple cubic 128^3 lattice (2,097,152 spins) the headline metric is quoted on.
    value   whole-job spin-updates/s, state resident in HBM, CUDA events on the launching stream, max over ranks
    e2e     the same through the C-ABI with HOST buffers: spins_set(host) + llg_iterate + spins_get(host) per step
    roofline dominant kernel (corrector): algorithmic bytes per launch / its live duration, against the measured HBM peak
    cpu_baseline  the oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample (rank 0, N=1)
N > 1: replicas only (the path has no exchange step on one GPU per lattice): every rank advances
its own lattice, no data-path collective, weak scaling.
`--impl reference` times the oracle alone (the reference arm of this tier).
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
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

ALG_BYTES_PREDICTOR = 48    # read n (24 B) + write n^p (24 B) per spin
ALG_BYTES_CORRECTOR = 72    # read n^p, read n, write n (24 B each) per spin; A recomputed
ALG_BYTES_STEP = ALG_BYTES_PREDICTOR + ALG_BYTES_CORRECTOR


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            p = json.load(open(path))
            return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def committed_traffic(workload):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture (profiles/), or None."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    try:
        return json.load(open(path)).get(workload, {}).get("corrector_dram_bytes_per_launch")
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0, period_ms=200):
        self.index = index
        self.period_ms = int(period_ms)
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", str(self.period_ms)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for k, nm in enumerate(names) if any(len(r) >= 7 and r[3 + k].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm), "power_w_max": max(pw) if pw else None}


def oracle_rate(w, budget_s=12.0, threads=None):
    """Time the oracle, as it stands, on a bounded sample of workload `w`: spin-updates/s on the host cores."""
    import oracle
    o = oracle.OracleSystem.from_workload(w)
    if threads:
        o.set_threads(threads)
    t0 = time.perf_counter()
    o.iterate(1)
    t1 = time.perf_counter() - t0
    n = int(max(1, min(200, budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter()
    o.iterate(n)
    dt = time.perf_counter() - t0
    return w.n_spins * n / dt, o.threads, f"{w.name}: {n} Depondt iterations of the full lattice ({w.n_spins} spins), {dt:.1f} s"


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    sample = ""
    cores = 0
    for _ in range(args.warmup):
        oracle_rate(w, budget_s=1.0)
    t_all = time.perf_counter()
    for _ in range(args.steps):
        v, cores, sample = oracle_rate(w, budget_s=max(2.0, 60.0 / max(args.steps, 1)))
        vals.append(v)
    wall = time.perf_counter() - t_all
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": "spin-updates/sec (fp64 LLG Depondt iterations x spins)", "value": value, "unit": "spin-updates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "spins": w.n_spins, "note": "CPU oracle on host cores; each step is a bounded sample"},
        "cpu_baseline": {"value": value, "unit": "spin-updates/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "spin-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number (1-5); default 3 = 128^3 headline")
    ap.add_argument("--inner", type=int, default=128, help="LLG iterations per bench step (a multiple of the 16-step CUDA graph)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--store-A", type=int, default=0)
    ap.add_argument("--clock-period-ms", type=int, default=200, help="nvidia-smi sampling period during the timed region (the recipe's 200 ms)")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE", help="spin_set_option pass-through (e.g. use_pdl=0) for A/B runs")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = W.CONFIGS[args.config]()

    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    import paper_1901_11350_b200 as P

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_1901_11350_b200 import replicas
    w = replicas.replica_workload(w, rank)          # N > 1: independent replicas, one per rank (no data-path collective)
    stream = torch.cuda.Stream()
    n0 = w.initial_spins()
    sys_ = P.SpinSystem.from_workload(w, stream=stream.cuda_stream)
    sys_.spin_set_option("store_A", args.store_A)
    for kv in args.option:
        name, value = kv.split("=")
        sys_.spin_set_option(name, int(value))
    N = sys_.N
    inner = args.inner

    # ---------------- device-resident timing
    # the clock sampler starts before the warm-up and the timed steps follow the warm-up without an idle gap: after idling the board
    # runs the first 40 ms about 8 % faster than in its steady state, and a pause here would time mostly that
    sampler = ClockSampler(local, args.clock_period_ms)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            sys_.llg_iterate(inner)
    barrier()
    l0, f0 = sys_.spin_launch_counts()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(args.steps):
            sys_.llg_iterate(inner)
        ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    l1, f1 = sys_.spin_launch_counts()
    clocks = sampler.stop() if rank == 0 else None
    ms_max = replicas.max_over_ranks(ms, device="cuda")
    value = replicas.whole_job_rate(N, inner * args.steps, ms_max, world)

    # ---------------- end to end through host buffers (pinned), copies inside the timed region
    host_in = torch.from_numpy(n0.copy()).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        sys_.spins_set(host_in.numpy()); sys_.llg_iterate(inner); sys_.spins_get(host_out.numpy())
    barrier()
    ee0, ee1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ee0.record(stream)
    for _ in range(e2e_steps):
        sys_.spins_set(host_in.numpy())
        sys_.llg_iterate(inner)
        sys_.spins_get(host_out.numpy())
    ee1.record(stream)
    barrier()
    e2e_ms = ee0.elapsed_time(ee1)      # events on the launching stream bracket copies + kernels; the host blocks on each copy
    e2e_value = replicas.whole_job_rate(N, inner * e2e_steps, replicas.max_over_ranks(e2e_ms, device="cuda"), world)

    # ---------------- per-kernel split (events around every launch, plain launches) -> live duration of the dominant kernel
    sys_.spin_profile_enable(True)
    sys_.llg_iterate(50)
    sys_.spin_synchronize()
    p_ms, p_n = sys_.spin_profile_get(0)
    c_ms, c_n = sys_.spin_profile_get(1)
    d_ms, d_n = sys_.spin_profile_get(2)
    sys_.spin_profile_enable(False)
    per_iter = {"predictor": p_ms / max(p_n, 1), "corrector": c_ms / max(c_n, 1), "ddi": 2 * d_ms / max(d_n, 1) if d_n else 0.0}
    tot = sum(per_iter.values())
    ms_per_iter = ms_max / (inner * args.steps)
    corr_live_ms = ms_per_iter * per_iter["corrector"] / tot            # share from the profiled pass x live time per iteration
    peak, peak_src = measured_peaks()
    fp64_tflops = sys_.spin_measure_fp64_tflops()       # the ALU ceiling: the path sits near the fp64 ridge (about 5 flop/B)
    achieved = ALG_BYTES_CORRECTOR * N / (corr_live_ms * 1e-3) / 1e9
    step_gbs = ALG_BYTES_STEP * N / (ms_per_iter * 1e-3) / 1e9

    if rank == 0:
        line = {
            "metric": "spin-updates/sec (fp64 LLG Depondt iterations x spins)", "value": value, "unit": "spin-updates/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "spins": N, "llg_iterations_per_step": inner, "solver": "Depondt", "parallelism": f"replicas x{world}",
                       "l2": "state arrays n, n^p, n' = %.0f MB > 126 MB L2 (no flush needed)" % (3 * 24 * N / 1e6) if 72 * N > 126e6 else
                             "state %.1f MB is L2-resident; effective bandwidth reported" % (3 * 24 * N / 1e6),
                       "store_A": args.store_A, "kernels": sys_.spin_kernel_info(), "ddi": sys_.spin_ddi_info(), "nvrtc": P.spin_jit_compiler_info()},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "spin-updates/s", "h2d_bytes_per_step": int(host_in.numel() * 8), "d2h_bytes_per_step": int(host_out.numel() * 8),
                    "steps": e2e_steps},
            "gpu_launches": int(l1 - l0), "cufft_execs": int(f1 - f0),
            "roofline": {"bound": "hbm", "kernel": "jit_corrector" if sys_.spin_kernel_info().startswith("jit") else "corrector_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "peak_source": peak_src, "traffic": committed_traffic(w.name),
                         "algorithmic_bytes_per_launch": ALG_BYTES_CORRECTOR * N, "launch_ms": corr_live_ms,
                         "kernel_share_of_step": per_iter["corrector"] / tot,
                         "step_effective_gbs": step_gbs, "step_frac_of_peak": step_gbs / peak, "step_frac_of_8000": step_gbs / 8000.0,
                         "profiled_ms": per_iter,
                         # fp64 instructions per spin-update counted by ncu on cfg3 (profiles/r1e): 77 + 130 warp instructions of 32 lanes
                         "fp64_peak_tflops_measured": fp64_tflops,
                         "fp64_frac_cfg3_count": (2.0 * 207 * N / (ms_per_iter * 1e-3) / 1e12) / fp64_tflops if w.name.startswith("cfg3") else None},
        }
        if world == 1 and not args.no_cpu_baseline:
            v, cores, sample = oracle_rate(w)
            line["cpu_baseline"] = {"value": v, "unit": "spin-updates/s", "cores": cores, "kind": "oracle", "sample": sample}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
