#!/usr/bin/env python
"""bench.py -- throughput of the fused viscous KT-RK2 step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--precision 64|32] [--kernel 0|1|2|3|4]
    python bench.py --impl reference ...      # the CPU oracle, timed as it stands (bounded sample per step)

A "step" is one full RK2 step (both stages: KT fluxes of T^{tau mu} and pi^{mu nu} on three axes, Milne and
Israel-Stewart sources, root-find, pi limiter, reductions) over the whole grid.  Workload = BASELINE.json
configs[4]: 301x301x201 cells, dx=dy=0.1, deta=0.08, tau0=0.4, dtau=0.01, eta/s=0.16, crossover EoS table,
8000 seeded partons with momentum (synthetic stand-in for AMPT events).  Prints ONE JSON line: the headline is
the fp64 run (BASELINE.json's metric names fp64 and fp32; the fp32 run of the same grid and step count is the
"fp32" sub-record of the same line).

Timing: W >= 3 warm-up steps, then exactly K steps between CUDA events recorded on the stream the
kernels are launched on, stream-synchronised on both sides (barrier + max over ranks for N > 1).  The
working set (3 state buffers of 14-19 fields x 146 MB) is far larger than the 126 MB L2, so no flush is needed.
N > 1: one process per GPU, each evolving its own seeded event (replicas, no data-path collective; "scaling": "weak");
`--decomp slabs` instead splits ONE event into eta_s slabs with a ghost-plane exchange after each stage ("strong").
`--gpus N` without a torchrun environment re-executes itself under torch.distributed.run.
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
ALGO_WORDS = {True: 73, False: 20}     # compulsory words per cell per RK2 step (viscous / ideal)
NSM, ISSUE_PER_SM = 148, 4             # B200: SMs, warp-instruction issue slots per clock per SM (4 schedulers)


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_counters():
    """Per-launch counters of the stage kernels taken from the committed ncu captures (profiles/round2_counters.json):
    dram bytes and executed warp instructions, keyed f<precision>_k<kernel>."""
    p = os.path.join(ROOT, "profiles", "round2_counters.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f)
    return {}


class ClockSampler(threading.Thread):
    """SM clock / throttle reasons during the run: one long-lived `nvidia-smi -lms 50` (B200_PROFILING.md recipe),
    started before the warm-up; every line is stamped when it is read."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0, period_ms=50):
        super().__init__(daemon=True)
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", str(period_ms)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, bufsize=1)
        except Exception:
            self.proc = None

    def run(self):
        if not self.proc:
            return
        for line in self.proc.stdout:
            self.rows.append([time.perf_counter()] + [c.strip() for c in line.strip().split(",")])

    def stop(self, windows):
        """windows: list of (t0, t1) perf_counter intervals of the timed regions."""
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
        self.join(timeout=5)
        inside = [r[1:] for r in self.rows if any(t0 <= r[0] <= t1 for t0, t1 in windows)]
        sm, reasons, mx = [], set(), None
        for r in (inside or [r[1:] for r in self.rows]):
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        ts = [r[0] for r in self.rows]
        period = 1e3 * float(np.median(np.diff(ts))) if len(ts) > 2 else None     # what nvidia-smi really delivered
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(self.rows), "samples_inside_timed_region": len(inside), "period_ms_requested": 50,
                "period_ms_measured": period}


def sub_config(nx, ny, nz, partons):
    """A sub-box of configs[4]: same spacings, times, eta/s, EoS and sampler; fewer cells / partons."""
    c = inputs.config4(nx=nx, ny=ny, nz=nz)
    c.extra = {"partons": partons, "moving": True}
    return c


def make_oracle(nx, ny, nz):
    from oracle import Oracle
    full = (nx, ny, nz) == (301, 301, 201)
    partons = 8000 if full else max(8, int(round(8000 * nx * ny * nz / (301.0 * 301 * 201))))
    cfg = sub_config(nx, ny, nz, partons)
    eos = inputs.crossover_table()
    T, _ = inputs.ic_partons(cfg, inputs.seed_for(4))
    o = Oracle(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.deta, cfg.dtau, cfg.tau0, eos, cfg.eta_over_s)
    o.load(T)
    what = ("configs[4] itself (301x301x201, 8000 partons)" if full else
            f"{nx}x{ny}x{nz} sub-box of configs[4] (same spacings, EoS table, eta/s=0.16, sampler at the same parton "
            f"density: {partons} partons)")
    return o, cfg, what


def omp_threads():
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores.  Every step of the run is one RK2 step of a bounded
    sample (a 96x96x64 sub-box of configs[4]); W warm-up steps, then exactly K timed steps."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    o, cfg, what = make_oracle(96, 96, 64)
    o.step(max(args.warmup, 0))
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    rate = cfg.cells * args.steps / dt
    sample = f"{what}; {args.steps} RK2 steps after {args.warmup} warm-up steps, {dt:.1f} s wall"
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[4] 301x301x201 viscous eta/s=0.16 crossover EoS; the oracle is timed on a "
                                   "bounded sample of it per step", "sample": sample, "cells_per_step": cfg.cells},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": omp_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def roofline_record(cells, precision, viscous, ms_total, launches, kernel, counters, clocks):
    """The dominant kernel is the stage kernel (two launches per step, 100 % of hydro_step)."""
    peak, peak_src = measured_hbm_peak()
    algo_per_launch = ALGO_WORDS[viscous] * (precision // 8) * cells / 2.0
    avg_launch_s = ms_total * 1e-3 / launches
    achieved = algo_per_launch / avg_launch_s / 1e9
    c = counters.get(f"f{precision}_k{kernel}", {}) if viscous else {}
    rec = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
           "traffic": c.get("dram_bytes_per_launch"), "peak_source": peak_src,
           "kernel": {1: "stage_ref_kernel", 2: "stage_fused_kernel", 3: "stage_tile_kernel", 4: "stage_march_kernel"}[kernel] +
                     " (average of the stage-1 and stage-2 launches)",
           "algorithmic_bytes_per_launch": algo_per_launch, "avg_launch_ms": avg_launch_s * 1e3}
    # second view: what actually limits the kernel is instruction issue / fp64 latency, not HBM.
    # Measured warp instructions per launch (ncu, profiles/) over the issue slots available during the measured launch.
    wi = c.get("warp_inst_per_launch")
    if wi:
        sm_hz = 1e6 * ((clocks or {}).get("sm_mhz") or 1965.0)
        rec["issue"] = {"bound": "alu", "achieved": wi / avg_launch_s, "peak": NSM * ISSUE_PER_SM * sm_hz,
                        "unit": "warp-inst/s", "frac": wi / avg_launch_s / (NSM * ISSUE_PER_SM * sm_hz),
                        "source": c.get("source")}
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--precision", type=int, default=64, choices=(64, 32),
                    help="precision of the headline run (default 64; the other precision is the sub-record)")
    ap.add_argument("--kernel", type=int, default=0)
    ap.add_argument("--impl", default="b200", choices=("b200", "reference"))
    ap.add_argument("--decomp", default="replicas", choices=("replicas", "slabs"),
                    help="N > 1: one seeded event per rank (default, weak scaling, no data-path communication) or ONE "
                         "event split into eta_s slabs with a ghost-plane exchange after each stage (strong scaling)")
    ap.add_argument("--grid", default="301,301,201", help="nx,ny,nz (default = configs[4])")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-steps", type=int, default=3, help="oracle steps of configs[4] for cpu_baseline (0 = skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-second-precision", action="store_true")
    ap.add_argument("--eta-over-s", type=float, default=0.16,
                    help="context runs only (0 = the ideal-fluid path, PAPER.md Table II); the headline is 0.16")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "RANK" not in os.environ:
        # launched by hand without torchrun: start one rank per GPU ourselves
        port = str(29500 + os.getpid() % 2000)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", port, os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
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
    slab_mode = args.decomp == "slabs" and world > 1
    # replicas: one seeded event per rank; slabs: every rank cuts its planes out of the same event
    T, _ = inputs.ic_partons(cfg, replicas.rank_seed(4, 0 if slab_mode else rank))
    viscous = args.eta_over_s > 0
    counters = ncu_counters()

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    windows = []

    def timed_run(precision):
        """Device-resident timing of K steps in one precision; returns the context and the record."""
        npdt = np.float64 if precision == 64 else np.float32
        if slab_mode:
            from paper_1802_04449_b200 import slabs
            sl = slabs.Slab(cfg, eos, rank, world, precision=precision, kernel=args.kernel, device=f"cuda:{local}")
            sl.load(T)
            h = sl.h
            step = lambda n: sl.step(n, slabs.exchange_dist)
        else:
            h = from_config(cfg, eos, precision=precision, kernel=args.kernel, device=f"cuda:{local}")
            h.load(torch.from_numpy(T.astype(npdt)).to(dev))
            step = h.step
        step(args.warmup)
        barrier()
        l0 = h.launch_count()
        tw0 = time.perf_counter()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(h.stream)
        step(args.steps)
        ev1.record(h.stream)
        barrier()
        windows.append((tw0, time.perf_counter()))
        ms_local = ev0.elapsed_time(ev1)
        launches = h.launch_count() - l0
        # slabs: the N ranks share ONE event (cells of the whole grid once); replicas: N events
        value, ms = replicas.aggregate_rate(cfg.cells / world if slab_mode else cfg.cells, args.steps, ms_local, world, dev)
        return h, dict(value=value, ms=ms, launches=int(launches), kernel=h.kernel(), diag=h.diag())

    h, main_rec = timed_run(args.precision)

    # ---- end to end through the C ABI with HOST buffers (pinned): load -> step -> read, every step ------
    N = cfg.cells
    npdt = np.float64 if args.precision == 64 else np.float32
    tdt = torch.float64 if args.precision == 64 else torch.float32
    T_host = torch.from_numpy(T.astype(npdt)).pin_memory()
    e_h = torch.empty((nz, ny, nx), dtype=tdt, pin_memory=True)
    u_h = torch.empty((4, nz, ny, nx), dtype=tdt, pin_memory=True)

    def e2e_step():
        h.load(T_host)
        h.step(1)
        h.read(out=(e_h, u_h, None))      # the method's result: e and u^mu

    e2e = None
    if args.e2e_steps > 0 and not slab_mode:
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e2e_step()
        barrier()
        e2e_s = replicas.max_over_ranks(max(time.perf_counter() - t0, 1e-9), dev)
        esz = 8 if args.precision == 64 else 4
        e2e = {"value": world * N * args.e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 4 * N * esz,
               "d2h_bytes_per_step": 5 * N * esz, "steps": args.e2e_steps,
               "what": "hydro_load(host T^{tau mu}) + hydro_step(1) + hydro_read(host e, u^mu) per step, pinned buffers; "
                       "pi^{mu nu} is neither loaded (initial pi = 0, as in configs[4]) nor read back: a viscous restart "
                       "would copy 10 more words per cell each way"}
    del h

    # ---- the other precision of BASELINE.json's metric, same grid and step count -------------------------
    second = None
    if not args.no_second_precision:
        p2 = 32 if args.precision == 64 else 64
        h2, second = timed_run(p2)
        second["precision"] = p2
        del h2

    clocks = sampler.stop(windows) if sampler else None
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    roofline = roofline_record(cfg.cells, args.precision, viscous, main_rec["ms"], main_rec["launches"],
                               main_rec["kernel"], counters, clocks)
    second_rec = None
    if second:
        p2 = second["precision"]
        second_rec = {"dtype": f"f{p2}", "value": second["value"], "unit": UNIT, "steps": args.steps,
                      "ms_per_step": second["ms"] / args.steps, "kernel": second["kernel"],
                      "gpu_launches": second["launches"],
                      "roofline": roofline_record(cfg.cells, p2, viscous, second["ms"], second["launches"],
                                                  second["kernel"], counters, clocks),
                      "diag": {k: second["diag"][k] for k in ("tau", "step", "e_max", "nan", "root_unconverged")}}

    cpu = None
    if not args.no_cpu_baseline and world == 1 and args.cpu_steps > 0:      # rank 0 at N = 1 only
        full = (nx, ny, nz) == (301, 301, 201)
        o, ocfg, what = make_oracle(nx, ny, nz) if full else make_oracle(96, 96, 64)
        t0 = time.perf_counter()
        o.step(args.cpu_steps)
        dt = time.perf_counter() - t0
        cpu = {"value": ocfg.cells * args.cpu_steps / dt, "unit": UNIT, "cores": omp_threads(), "kind": "oracle",
               "sample": f"{what}, {args.cpu_steps} RK2 steps, {dt:.1f} s wall (load and bootstrap not timed)"}
        del o

    d = main_rec["diag"]
    line = {"metric": METRIC, "value": main_rec["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main_rec["ms"] / args.steps, "higher_is_better": True,
            "scaling": "strong" if slab_mode else "weak", "vs_baseline": None,
            "dtype": "f64" if args.precision == 64 else "f32",
            "data": "synthetic",
            "config": {"workload": f"configs[4]: {nx}x{ny}x{nz} cells, dx=dy=0.1 fm, deta=0.08, tau0=0.4, dtau=0.01, "
                                   f"eta/s={args.eta_over_s:g}, crossover EoS table (2000 nodes), {cfg.extra['partons']} seeded "
                                   "partons with momentum, outflow boundaries",
                       "cells": cfg.cells, "precision": args.precision, "kernel": main_rec["kernel"],
                       "kernel_requested": args.kernel,
                       "l2": "working set (3 state buffers) >> 126 MB L2, no flush needed",
                       "parallelism": ("1 event in %d eta_s slabs, ghost-plane exchange after each stage (NCCL send/recv)" % world
                                       if slab_mode else ("1 event per GPU (replicas)" if world > 1 else "1 GPU"))},
            "roofline": roofline, "fp32" if args.precision == 64 else "fp64": second_rec,
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": main_rec["launches"], "clocks": clocks,
            "diag": {k: d[k] for k in ("tau", "step", "cfl", "e_max", "floored", "clamped", "pi_limited", "nan",
                                       "root_unconverged")},
            "context": {"paper": "CLVisc: 16.9 M cell-updates/s viscous fp32 on AMD FirePro S9150 (Table II, "
                                 "PAPER.md:646-654); ~60x evolution speed-up vs one CPU core (PAPER.md:21)"}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
