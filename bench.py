#!/usr/bin/env python
"""bench.py -- spin-updates/s of the LLG hot path on B200 (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--min-seconds 2.0]

One bench "step" = one `llg_iterate(inner)` call = `inner` Depondt iterations (each: field of every spin at n, predictor, field at
n^p, corrector; all rows of SURVEY 8(a)) over the whole lattice.  `inner` is a multiple of the 16-step CUDA graph, chosen during the
warm-up so that the K timed steps last at least --min-seconds (2 s): the board needs about 0.1 s under this load to settle at its
1000 W power cap, and the clock sampler needs the load to last (a run of 0.2 s times mostly the faster first 40 ms).
Workload at N=1: configs[2] of BASELINE.json, the 3-D simple cubic 128^3 lattice (2,097,152 spins) the headline metric is quoted on.
    value    whole-job spin-updates/s, state resident in HBM, CUDA events on the launching stream, max over ranks
    e2e      the same through the C-ABI with HOST buffers: spins_set(host) + llg_iterate(128) + spins_get(host) per step
    roofline the dominant kernel OF THE WORKLOAD: algorithmic bytes per launch / its live duration, against the measured HBM peak
    configs  the other four BASELINE.json workloads: throughput, us per Depondt step, roofline of their dominant kernel, and the
             residual of a short trajectory against the oracle at full size (rank 0, N=1; --no-configs skips them)
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

# Algorithmic bytes per spin and launch (fp64 SoA, 24 B per spin and array; neighbour reads are cache hits):
#   predictor: read n, write n^p (+ write the thermal field of the step when T > 0 and cache_noise is on)
#   corrector: read n^p, read n, write n(t+dt) (+ read the thermal field)
def sweep_bytes(thermal: bool):
    return (72, 96) if thermal else (48, 72)


def ddi_contract_bytes(w):
    """Algorithmic bytes of one launch of the dipolar contraction kernel on the slab path: the spectra of the 3 NZ
    slabs are read and written in place (16 B per in-plane wave vector and slab, twice), the real 6-component tensor is read at
    PZ / 2 + 1 planes along c (mirror symmetric spectrum) of the PZ = 2 NZ."""
    na, nb, nz = w.n_cells
    s2 = (2 * nb) * (na + 1)                      # in-plane wave vectors of the half spectrum: P1 * (P0 / 2 + 1)
    pz = 2 * nz if nz > 1 else 1
    return s2 * (2 * 16 * 3 * nz + 6 * 8 * (pz // 2 + 1))


def ddi_fused_bytes(w, mirror=True):
    """Algorithmic bytes of one launch of the fused b-pass kernel: the a-pass spectra [ka][slab][ib] are read once
    (16 B per element), the real 6-component tensor is read at NZ + 1 (mirror symmetric) or 2 NZ planes for every in-plane wave vector,
    and the two partial results (one per parity of kb) are written."""
    na, nb, nz = w.n_cells
    s1 = na + 1                                   # wave numbers along a of the half spectrum: P0 / 2 + 1
    planes = nz + 1 if mirror else 2 * nz
    return s1 * nb * (16 * 3 * nz + 2 * 16 * 3 * nz) + s1 * 2 * nb * 6 * 8 * planes


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            p = json.load(open(path))
            return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def committed_traffic(workload, kernel):
    """dram bytes per launch of `kernel` on `workload` from the committed ncu captures (profiles/roofline_traffic.json), or None."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    try:
        return json.load(open(path)).get(workload, {}).get(kernel)
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


def workload_config(w, world):
    """The `config` object of the JSON line: what the workload IS.  Both arms (ours / reference) emit exactly this for the same workload;
    how a run was carried out (iterations per step, kernels, compiler) goes into `run`."""
    return {"workload": w.name, "spins": int(w.n_spins), "solver": "Depondt", "cells": list(map(int, w.n_cells)),
            "periodic": list(map(int, w.periodic)), "parallelism": f"replicas x{world}"}


def measure_workload(P, torch, w, stream, steps, warmup, min_seconds, barrier=None, options=(), store_A=0, e2e=True, reducer=None):
    """Device-resident throughput of workload `w` on the current device, its e2e figure and the roofline of its dominant kernel.
    Returns (system, dict).  `reducer(ms)` turns the local device time into the max over ranks (identity by default)."""
    barrier = barrier or torch.cuda.synchronize
    reducer = reducer or (lambda ms: ms)
    sys_ = P.SpinSystem.from_workload(w, stream=stream.cuda_stream)
    sys_.spin_set_option("store_A", store_A)
    for kv in options:
        name, value = kv.split("=")
        sys_.spin_set_option(name, int(value))
    N = sys_.N
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # ---------------- warm-up, and the number of iterations per step that makes the timed region last min_seconds
    with torch.cuda.stream(stream):
        sys_.llg_iterate(128)
        ev0.record(stream)
        sys_.llg_iterate(256)
        ev1.record(stream)
    barrier()
    us_iter = reducer(ev0.elapsed_time(ev1)) * 1e3 / 256
    inner = int(max(128, -(-min_seconds * 1e6 / max(steps, 1) / us_iter // 16) * 16))
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            sys_.llg_iterate(inner)
    barrier()
    l0, f0 = sys_.spin_launch_counts()
    barrier()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(steps):
            sys_.llg_iterate(inner)
        ev1.record(stream)
    barrier()
    ms = reducer(ev0.elapsed_time(ev1))
    l1, f1 = sys_.spin_launch_counts()
    out = {"N": N, "inner": inner, "ms": ms, "ms_per_iter": ms / (inner * steps), "gpu_launches": int(l1 - l0), "cufft_execs": int(f1 - f0)}

    # ---------------- end to end through host buffers (pinned), copies inside the timed region
    if e2e:
        n0 = w.initial_spins()
        host_in = torch.from_numpy(n0.copy()).pin_memory()
        host_out = torch.empty_like(host_in).pin_memory()
        e2e_inner, e2e_steps = 128, max(3, min(steps, 10))
        for _ in range(2):
            sys_.spins_set(host_in.numpy()); sys_.llg_iterate(e2e_inner); sys_.spins_get(host_out.numpy())
        barrier()
        ee0, ee1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ee0.record(stream)
        for _ in range(e2e_steps):
            sys_.spins_set(host_in.numpy())
            sys_.llg_iterate(e2e_inner)
            sys_.spins_get(host_out.numpy())
        ee1.record(stream)
        barrier()
        out["e2e"] = {"ms": reducer(ee0.elapsed_time(ee1)), "inner": e2e_inner, "steps": e2e_steps, "h2d": int(host_in.numel() * 8), "d2h": int(host_out.numel() * 8)}

    # ---------------- per-kernel split (events around every launch, plain launches) -> live duration of the dominant kernel
    kinfo, dinfo = sys_.spin_kernel_info(), sys_.spin_ddi_info()
    thermal = w.T > 0
    bp, bc = sweep_bytes(thermal and store_A == 0)
    if store_A:
        bp, bc = 72, 96                     # A(n) written by the predictor and read back by the corrector
    sys_.spin_profile_enable(True)           # (this also takes the lattice off the all-steps-in-one-launch path)
    sys_.llg_iterate(50)
    sys_.spin_synchronize()
    prof = [sys_.spin_profile_get(k) for k in range(4)]
    sys_.spin_profile_enable(False)
    per_iter = {"predictor": prof[0][0] / max(prof[0][1], 1), "corrector": prof[1][0] / max(prof[1][1], 1),
                "ddi": 2 * prof[2][0] / max(prof[2][1], 1) if prof[2][1] else 0.0,
                "ddi_contract": 2 * prof[3][0] / max(prof[3][1], 1) if prof[3][1] else 0.0}
    tot = per_iter["predictor"] + per_iter["corrector"] + per_iter["ddi"]
    peak, peak_src = measured_peaks()
    ms_iter = out["ms_per_iter"]
    step_bytes = (bp + bc) * N
    roof = {"bound": "hbm", "peak": peak, "unit": "GB/s", "peak_source": peak_src, "profiled_ms": per_iter,
            "step_algorithmic_bytes": step_bytes, "step_effective_gbs": step_bytes / (ms_iter * 1e-3) / 1e9}
    if dinfo.startswith("slab") and per_iter["ddi_contract"] > 0:
        # dipolar workloads: the evaluations are most of the step; their longest kernel is the fused b-pass (transforms along b and c, the
        # contraction and their inverses) or, without it, the contraction kernel; two launches per Depondt iteration
        if "fused-b" in dinfo:
            kernel, nbytes = "ddi_bfused_kernel", ddi_fused_bytes(w, "mirror" in dinfo)
            roof["note"] = ("dominant kernel of the dipolar evaluation (fused b-pass + c-pass + contraction); two launches per Depondt "
                            "iteration; fp64 issue and load latency co-limit it (profiles/r2_README.md)")
        else:
            kernel, nbytes = "ddi_slab_contract_kernel", ddi_contract_bytes(w)
            roof["note"] = "dominant kernel of the dipolar evaluation (cuFFT's b-passes are library kernels); two launches per Depondt iteration"
        # the kernel's own duration: CUDA events around it alone on the library's stream (profile mode; it runs between two host
        # synchronisations there, so nothing overlaps it); its share of the timed step follows from that
        launch_ms = per_iter["ddi_contract"] / 2
        share = min(1.0, 2 * launch_ms / ms_iter)
    elif "march" in kinfo:
        # the whole Depondt step is ONE kernel (n^p never leaves the SM): one launch = one iteration.  The roofline figure stays the method's
        # 120 B per spin-update (read n, write n^p; read n^p, read n, write n); the kernel's own DRAM traffic (`traffic`, about
        # 43 B per spin-update) is lower because it skips the n^p round trip and the second read of n.
        step_bytes = 120 * N                 # (the thermal field costs the method no traffic: regenerated from counters)
        roof["step_algorithmic_bytes"], roof["step_effective_gbs"] = step_bytes, step_bytes / (ms_iter * 1e-3) / 1e9
        kernel, nbytes = "jit_depondt_march", step_bytes
        share, launch_ms = 1.0, ms_iter
        roof["note"] = "one-pass plane-marching kernel: one launch per Depondt iteration; algorithmic bytes of the two-sweep method (120 B per spin-update)"
    elif "cluster" in kinfo or "coop" in kinfo:
        # launch-bound lattices: all steps in one launch, the state (24 KB-100 KB) never leaves L2; the figure is the effective bandwidth of
        # a step and says how far from HBM-bound the workload is, not how good the kernel is (its bound is the barrier latency)
        kernel, nbytes = ("jit_steps_cluster" if "cluster" in kinfo else "jit_steps_coop"), step_bytes
        share, launch_ms = 1.0, ms_iter
        roof["note"] = "all steps in one launch; per-iteration figure; latency-bound (two barriers per iteration), state L2-resident"
    else:
        kernel, nbytes = ("jit_corrector" if kinfo.startswith("jit") else "corrector_kernel"), bc * N
        share = per_iter["corrector"] / tot
        launch_ms = ms_iter * share
        if 3 * 24 * N < 126e6:
            roof["note"] = "state %.1f MB is L2-resident: effective bandwidth" % (3 * 24 * N / 1e6)
    roof.update({"kernel": kernel, "algorithmic_bytes_per_launch": int(nbytes), "launch_ms": launch_ms, "kernel_share_of_step": share,
                 "achieved": nbytes / (launch_ms * 1e-3) / 1e9, "traffic": committed_traffic(w.name.split("#")[0], kernel)})
    roof["frac"] = roof["achieved"] / peak
    roof["step_frac_of_peak"] = roof["step_effective_gbs"] / peak
    roof["step_frac_of_8000"] = roof["step_effective_gbs"] / 8000.0
    out["roofline"] = roof
    out["kernels"], out["ddi"] = kinfo, dinfo
    return sys_, out


def short_parity(P, w, steps):
    """max |n_gpu - n_oracle| after `steps` Depondt iterations of the full-size workload from its seeded start (oracle on the host cores)."""
    import oracle
    g = P.SpinSystem.from_workload(w)
    o = oracle.OracleSystem.from_workload(w)
    g.llg_iterate(steps)
    o.iterate(steps)
    d = float(np.abs(g.spins_get() - o.spins()).max())
    g.close()
    return d


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
        "config": workload_config(w, args.gpus),
        "run": {"note": "CPU oracle on host cores; each step is a bounded sample of the workload"},
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
    ap.add_argument("--min-seconds", type=float, default=2.0, help="least duration of the timed region (the iterations per step follow from it)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the other four workloads (the `configs` array)")
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

    # the clock sampler covers warm-up and timed region; the timed steps follow the warm-up without an idle gap
    sampler = ClockSampler(local, args.clock_period_ms)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    t_job = time.perf_counter()
    sys_, m = measure_workload(P, torch, w, stream, args.steps, args.warmup, args.min_seconds, barrier=barrier, options=args.option,
                               store_A=args.store_A, reducer=lambda ms: replicas.max_over_ranks(ms, device="cuda"))
    clocks = sampler.stop() if rank == 0 else None
    N, inner = m["N"], m["inner"]
    value = replicas.whole_job_rate(N, inner * args.steps, m["ms"], world)
    e = m["e2e"]
    e2e_value = replicas.whole_job_rate(N, e["inner"] * e["steps"], e["ms"], world)
    roof = m["roofline"]
    fp64_tflops = sys_.spin_measure_fp64_tflops()       # the ALU ceiling: the path sits near the fp64 ridge (about 5 flop/B)
    roof["fp64_peak_tflops_measured"] = fp64_tflops
    # fp64 instructions per spin-update counted by ncu on cfg3 (profiles/r1e): 77 + 130 warp instructions of 32 lanes
    roof["fp64_frac_cfg3_count"] = (2.0 * 207 * N / (m["ms_per_iter"] * 1e-3) / 1e12) / fp64_tflops if w.name.startswith("cfg3") else None

    if rank == 0:
        line = {
            "metric": "spin-updates/sec (fp64 LLG Depondt iterations x spins)", "value": value, "unit": "spin-updates/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": m["ms"] / args.steps,
            "us_per_llg_iteration": m["ms_per_iter"] * 1e3, "timed_region_s": m["ms"] * 1e-3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, world),
            "run": {"llg_iterations_per_step": inner,
                    "l2": ("state arrays n, n^p, n' = %.0f MB > 126 MB L2 (no flush needed)" % (3 * 24 * N / 1e6)) if 72 * N > 126e6 else
                          ("state %.1f MB is L2-resident; effective bandwidth reported" % (3 * 24 * N / 1e6)),
                    "store_A": args.store_A, "kernels": m["kernels"], "ddi": m["ddi"], "nvrtc": P.spin_jit_compiler_info()},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "spin-updates/s", "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"],
                    "steps": e["steps"], "llg_iterations_per_step": e["inner"]},
            "gpu_launches": m["gpu_launches"], "cufft_execs": m["cufft_execs"],
            "roofline": roof,
        }
        sys_.close()
        if world == 1 and not args.no_configs:
            # the other BASELINE.json workloads (north_star: throughput on the skyrmion, domain-wall and bobber shaped lattices): a shorter timed
            # region each, the roofline of their own dominant kernel, and a short trajectory against the oracle at full size
            parity_steps = {1: 200, 2: 50, 3: 8, 4: 20, 5: 4}
            configs = []
            for k in (1, 2, 3, 4, 5):
                if k == args.config:
                    continue
                wk = W.CONFIGS[k]()
                sk, mk = measure_workload(P, torch, wk, stream, 5, 3, 0.5, options=args.option, e2e=False)
                sk.close()
                rk = mk["roofline"]
                configs.append({"workload": wk.name, "spins": mk["N"], "value": mk["N"] * mk["inner"] * 5 / (mk["ms"] * 1e-3), "unit": "spin-updates/s",
                                "us_per_llg_iteration": mk["ms_per_iter"] * 1e3, "timed_region_s": mk["ms"] * 1e-3, "kernels": mk["kernels"], "ddi": mk["ddi"],
                                "roofline": {q: rk[q] for q in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "algorithmic_bytes_per_launch",
                                                                 "launch_ms", "kernel_share_of_step", "step_effective_gbs", "step_frac_of_peak") } | ({"note": rk["note"]} if "note" in rk else {}),
                                "parity": {"steps": parity_steps[k], "max_abs_dn_vs_oracle": short_parity(P, wk, parity_steps[k]), "tolerance": 1e-9}})
            line["configs"] = configs
        if world == 1 and not args.no_cpu_baseline:
            v, cores, sample = oracle_rate(w)
            line["cpu_baseline"] = {"value": v, "unit": "spin-updates/s", "cores": cores, "kind": "oracle", "sample": sample}
        line["wall_s"] = time.perf_counter() - t_job
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
