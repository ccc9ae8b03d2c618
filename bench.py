#!/usr/bin/env python
"""bench.py -- throughput of the fused viscous KT-RK2 step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--precision 64|32] [--kernel 0|1|2]
    python bench.py --impl reference ...      # the CPU oracle, timed as it stands (bounded sample)

A "step" is one full RK2 step (both stages: KT fluxes of T^{tau mu} and pi^{mu nu} on three axes, Milne and
Israel-Stewart sources, root-find, pi limiter, reductions) over the whole grid.  Workload = BASELINE.json
configs[4]: 301x301x201 cells, dx=dy=0.1, deta=0.08, tau0=0.4, dtau=0.01, eta/s=0.16, crossover EoS table,
8000 seeded partons with momentum (synthetic stand-in for AMPT events).  Prints ONE JSON line.

Timing: W >= 3 warm-up steps, then exactly K steps between CUDA events recorded on the stream the
kernels are launched on, stream-synchronised on both sides (barrier + max over ranks for N > 1).  The
working set (3 x 14 fields x 146 MB) is far larger than the 126 MB L2, so no flush is needed.
N > 1: one process per GPU, each evolving its own seeded event (replicas, no data-path collective).
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

from paper_1802_04449_b200 import inputs  # noqa: E402

METRIC = "viscous KT-RK2 cell-updates/s at 301x301x201"
UNIT = "cell-updates/s"
ALGO_BYTES_PER_CELL_STEP = {64: 584, 32: 292}     # 73 words per cell per RK2 step


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                if out.returncode == 0 and out.stdout.strip():
                    self.rows.append([time.perf_counter()] + [c.strip() for c in out.stdout.strip().split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self, t0=None, t1=None):
        self._stop_evt.set()
        self.join(timeout=10)
        sm, reasons, mx = [], set(), None
        inside = [r[1:] for r in self.rows if t0 is not None and t0 <= r[0] <= t1]
        for r in (inside or [r[1:] for r in self.rows]):
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm), "samples_inside_timed_region": len(inside)}


def sub_config(nx, ny, nz, partons):
    """A sub-box of configs[4]: same spacings, times, eta/s, EoS and sampler; fewer cells / partons."""
    c = inputs.config4(nx=nx, ny=ny, nz=nz)
    c.extra = {"partons": partons, "moving": True}
    return c


def cpu_oracle_rate(nx, ny, nz, steps):
    """Times the oracle as it stands on the host cores; returns (cell-updates/s, threads, description)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle import Oracle
    partons = max(8, int(round(8000 * nx * ny * nz / (301.0 * 301 * 201))))
    cfg = sub_config(nx, ny, nz, partons)
    eos = inputs.crossover_table()
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(4))
    o = Oracle(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.deta, cfg.dtau, cfg.tau0, eos, cfg.eta_over_s)
    o.load(T)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    sample = (f"{nx}x{ny}x{nz} sub-box of configs[4] (same spacings, EoS table, eta/s=0.16, sampler at the same "
              f"parton density: {partons} partons), {steps} RK2 step(s), {dt:.1f} s wall")
    return cfg.cells * steps / dt, threads, sample, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    nx, ny, nz = 96, 96, 64
    for _ in range(max(args.warmup, 0) and 1):
        cpu_oracle_rate(32, 32, 16, 1)
    rate, threads, sample, dt = cpu_oracle_rate(nx, ny, nz, max(1, min(args.steps, 4)))
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, min(args.steps, 4)),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[4] 301x301x201 viscous eta/s=0.16 crossover EoS; oracle timed on a bounded "
                                   "sample of it", "sample": sample},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--precision", type=int, default=64, choices=(64, 32))
    ap.add_argument("--kernel", type=int, default=0)
    ap.add_argument("--impl", default="b200", choices=("b200", "reference"))
    ap.add_argument("--grid", default="301,301,201", help="nx,ny,nz (default = configs[4])")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--eta-over-s", type=float, default=0.16,
                    help="context runs only (0 = the ideal-fluid path, PAPER.md Table II); the headline is 0.16")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_1802_04449_b200 import from_config, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CLVisc step has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    nx, ny, nz = [int(v) for v in args.grid.split(",")]
    cfg = inputs.config4(nx=nx, ny=ny, nz=nz, eta_over_s=args.eta_over_s)
    if (nx, ny, nz) != (301, 301, 201):
        cfg.extra["partons"] = max(8, int(round(8000 * cfg.cells / (301.0 * 301 * 201))))
    eos = inputs.crossover_table()
    T, _ = inputs.ic_partons(cfg, replicas.rank_seed(4, rank))     # one seeded event per rank
    npdt = np.float64 if args.precision == 64 else np.float32
    tdt = torch.float64 if args.precision == 64 else torch.float32

    h = from_config(cfg, eos, precision=args.precision, kernel=args.kernel, device=f"cuda:{local}")
    T_dev = torch.from_numpy(T.astype(npdt)).to(dev)
    h.load(T_dev)
    stream = h.stream

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    # ---- device-resident timing ----------------------------------------------------------------
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    h.step(args.warmup)
    barrier()
    l0 = h.launch_count()
    tw0 = time.perf_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    h.step(args.steps)
    ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = h.launch_count() - l0
    clocks = sampler.stop(tw0, time.perf_counter()) if sampler else None
    d = h.diag()
    value, ms = replicas.aggregate_rate(cfg.cells, args.steps, ms, world, dev)
    ms_per_step = ms / args.steps

    # ---- end to end through the C ABI with HOST buffers (pinned): load -> step -> read, every step ------
    N = cfg.cells
    T_host = torch.from_numpy(T.astype(npdt)).pin_memory()
    e_h = torch.empty((nz, ny, nx), dtype=tdt, pin_memory=True)
    u_h = torch.empty((4, nz, ny, nx), dtype=tdt, pin_memory=True)

    def e2e_step():
        h.load(T_host)
        h.step(1)
        h.read(out=(e_h, u_h, None))      # the method's result: e and u^mu

    if args.e2e_steps > 0:
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        e2e_step()
    barrier()
    e2e_s = max(time.perf_counter() - t0, 1e-9)
    e2e_s = replicas.max_over_ranks(e2e_s, dev)
    esz = 8 if args.precision == 64 else 4
    e2e = {"value": world * N * args.e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 4 * N * esz,
           "d2h_bytes_per_step": 5 * N * esz, "steps": args.e2e_steps,
           "what": "hydro_load(host T^{tau mu}) + hydro_step(1) + hydro_read(host e, u^mu) per step, pinned buffers"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the fused stage kernel: 2 launches per step) ------------------
    peak, peak_src = measured_hbm_peak()
    words = 73 if args.eta_over_s > 0 else 20            # compulsory words per cell per RK2 step
    algo_per_launch = words * (args.precision // 8) * cfg.cells / 2.0
    avg_launch_s = ms * 1e-3 / launches
    achieved = algo_per_launch / avg_launch_s / 1e9
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        with open(tp) as f:
            traffic = json.load(f).get(f"f{args.precision}_k{h_kernel_name(args.kernel)}")
    # second view: the same launch against the plain fp64 (fp32) pipe, 3 400 arithmetic
    # instructions per cell per stage on 148 SMs x 64 (128) lanes at the SM clock sampled during the run
    lanes = 64 if args.precision == 64 else 128
    sm_hz = 1e6 * ((clocks or {}).get("sm_mhz") or 1965.0)
    alu_frac = (3400.0 * cfg.cells / avg_launch_s) / (148 * lanes * sm_hz)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "alu_frac": alu_frac,
                "traffic": traffic, "peak_source": peak_src, "kernel": "fused RK2 stage kernel (avg of stage 1 and 2)",
                "algorithmic_bytes_per_launch": algo_per_launch, "avg_launch_ms": avg_launch_s * 1e3}

    cpu = None
    if not args.no_cpu_baseline and world == 1:      # rank 0 at N = 1 only
        rate, threads, sample, _ = cpu_oracle_rate(96, 96, 64, 2)
        cpu = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if args.precision == 64 else "f32", "data": "synthetic",
            "config": {"workload": f"configs[4]: {nx}x{ny}x{nz} cells, dx=dy=0.1 fm, deta=0.08, tau0=0.4, dtau=0.01, "
                                   f"eta/s={args.eta_over_s:g}, crossover EoS table (2000 nodes), {cfg.extra['partons']} seeded "
                                   "partons with momentum, outflow boundaries",
                       "cells": cfg.cells, "precision": args.precision, "kernel": args.kernel,
                       "l2": "working set (3 x 14 fields) >> 126 MB L2, no flush needed",
                       "parallelism": "1 event per GPU (replicas)" if world > 1 else "1 GPU"},
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
            "clocks": clocks,
            "diag": {k: d[k] for k in ("tau", "step", "cfl", "e_max", "floored", "clamped", "pi_limited", "nan",
                                       "root_unconverged")},
            "context": {"paper": "CLVisc: 16.9 M cell-updates/s viscous fp32 on AMD FirePro S9150 (Table II, "
                                 "PAPER.md:646-654); ~60x evolution speed-up vs one CPU core (PAPER.md:21)"}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def h_kernel_name(k):
    return {0: "default", 1: "ref", 2: "fused"}.get(k, str(k))


if __name__ == "__main__":
    main()
