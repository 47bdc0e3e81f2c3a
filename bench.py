#!/usr/bin/env python
"""bench.py -- particle-steps/s of the PIC-MC hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--scale 1.0] [--impl reference]

One "step" is one whole timestep (mover, side-list ordering + cell scan, arranger with fused deposit, field
solve) over every particle of the workload.  Default workload: BASELINE.json configs[3] (2e8 particles, 65536
cells, exponential sheath profile, 3 species, config-3 collisions) -- the first configuration at the
"1e8+ particles" size that the metric's HBM target is quoted on; configs[4] (1e9) also fits one GPU but its
host-side generation and load take several minutes (python bench.py --config 5 --steps 10 runs it).
Inputs are larger than L2 (8.2 GB state vs 126 MB), so no L2 flush is needed between steps.

Legs of one run: (1) W warm-up steps, then K timed steps bracketed by CUDA events on the compute stream (`value`;
bit1_step replays two-step CUDA graphs); (2) min(K, 50) more steps with CUDA events around every kernel (`roofline`);
(3) end to end: bit1_load_particles from pinned host arrays + K steps + bit1_get_rho to the host, wall clock (`e2e`);
(4) at N = 1, the CPU oracle on a bounded cut-down of the same workload (`cpu_baseline`).

The path does not shard (BASELINE.json north_star: no multi-GPU sharding or collectives): --gpus N runs N
independent replicas, one process per GPU, and reports the aggregate ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

STATE_BYTES = 41  # x, vx, vy, vz fp64 + cell int32 + pid uint32 + species uint8
METRIC = "particle-steps/sec"
UNIT = "particle-steps/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _traffic(kernel: str, args=None):
    """DRAM bytes per launch of the kernel from the committed ncu --set full capture (profiles/traffic.json);
    the capture is of the default workload, so any other workload reports null."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if args is not None and (args.config != 4 or args.scale != 1.0):
        return None
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f).get(kernel)
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows]
        for r in rows:
            f = [v.strip() for v in r.split(",")]
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
            except Exception:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def _dist():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def aggregate(local_ms: float, local_units: float, world: int, backend_device=None):
    """Max time over ranks and total units (replicas): the --gpus N reduction, also used by the gloo test."""
    if world == 1:
        return local_ms, local_units
    import torch
    import torch.distributed as dist

    t = torch.tensor([local_ms], dtype=torch.float64, device=backend_device)
    u = torch.tensor([local_units], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def _workload(args, rank: int):
    from paper_2606_28534_b200 import workloads as W

    w = W.make_config(args.config, scale=args.scale, gen_seed=2606285340 + args.config + 1000 * rank,
                      lib_seed=2606285340000 + args.config + 1000 * rank)
    name = f"BASELINE.json configs[{args.config - 1}]" + (f" cut down x{args.scale:g}" if args.scale != 1.0 else "")
    return w, name


def cpu_baseline(args, seconds_hint: float = 12.0):
    """The oracle as it stands, single thread, on a bounded cut-down of the same configuration."""
    from oracle.oracle import Oracle
    from paper_2606_28534_b200 import workloads as W

    target_n = 4.0e6
    full_n = {1: 204800, 2: 1638400, 3: 1e7, 4: 2e8, 5: 1e9}[args.config] * args.scale
    scale = args.scale * min(1.0, target_n / full_n)
    w = W.make_config(args.config, scale=scale)
    o = Oracle(w)
    o.step(1)
    steps = 0
    t0 = time.perf_counter()
    while True:
        o.step(2)
        steps += 2
        if time.perf_counter() - t0 > seconds_hint or steps >= 400:
            break
    dt = time.perf_counter() - t0
    return {"value": w.n * steps / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"configs[{args.config - 1}] cut down to {w.n} particles / {w.nc} cells (same particles per "
                      f"cell and profile), {steps} steps in {dt:.1f} s, single thread, gcc -O2 -ffp-contract=off"}


def run_reference(args):
    rank, world, _ = _dist()
    if rank != 0:
        return
    from oracle.oracle import Oracle
    from paper_2606_28534_b200 import workloads as W

    full_n = {1: 204800, 2: 1638400, 3: 1e7, 4: 2e8, 5: 1e9}[args.config] * args.scale
    scale = args.scale * min(1.0, 4.0e6 / full_n)
    w = W.make_config(args.config, scale=scale)
    o = Oracle(w)
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    val = w.n * args.steps / dt
    sample = (f"each step = one oracle timestep on configs[{args.config - 1}] cut down to {w.n} particles / {w.nc} "
              f"cells; single thread")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "particle-steps/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}] (bounded sample)", "particles": w.n,
                       "cells": w.nc},
            "cpu_baseline": {"value": val, "unit": "particle-steps/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "particle-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_cuda(args):
    import numpy as np
    import torch

    rank, world, local = _dist()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    from paper_2606_28534_b200.binding import Bit1

    w, wname = _workload(args, rank)
    n0 = w.n
    sim = Bit1(w, device=f"cuda:{local}")
    # pinned host copies of the inputs for the end-to-end leg
    pin = {}
    for k in ("x", "vx", "vy", "vz", "sp"):
        src = torch.from_numpy(getattr(w, k))
        try:
            pin[k] = src.pin_memory()
        except Exception:
            pin[k] = src
    h2d_bytes = sum(t.numel() * t.element_size() for t in pin.values())
    host = {k: t.numpy() for k, t in pin.items()}

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident leg: W warm-up steps, then exactly K timed steps ---------------------------
    sim.load_particles(host["x"], host["vx"], host["vy"], host["vz"], host["sp"])
    sim.step(args.warmup)
    sim.sync()
    n_start = sim.n_live()
    launches0 = sim.launch_count()
    ev0 = torch.cuda.Event(enable_timing=True)
    ev1 = torch.cuda.Event(enable_timing=True)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    t_wall0 = time.perf_counter()
    with torch.cuda.stream(sim.compute_stream):
        ev0.record(sim.compute_stream)
        sim.step(args.steps)
        ev1.record(sim.compute_stream)
    barrier()
    t_wall1 = time.perf_counter()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms = ev0.elapsed_time(ev1)
    launches = sim.launch_count() - launches0
    sim.sync()
    n_end = sim.n_live()
    units = 0.5 * (n_start + n_end) * args.steps
    # per-kernel leg (roofline): the same steps again with CUDA events around every kernel on the compute stream
    # (bit1_profile; direct launches -- the timed leg above replays two-step CUDA graphs)
    psteps_want = min(args.steps, 50)
    sim.profile(True)
    sim.step(psteps_want)
    prof, psteps = sim.get_profile()
    sim.profile(False)
    sim.sync()
    n_prof = 0.5 * (n_end + sim.n_live())
    ms_max, units_all = aggregate(ms, units, world, dev)
    mom = sim.get_moments()

    # ---- end-to-end leg: host buffers in, rho out, copies inside the timed region ----------------------
    barrier()
    t0 = time.perf_counter()
    sim.load_particles(host["x"], host["vx"], host["vy"], host["vz"], host["sp"])
    sim.step(args.steps)
    rho = sim.get_rho()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_ms_max, e2e_units = aggregate(1e3 * e2e_s, float(n0) * args.steps, world, dev)
    d2h_bytes = rho.nbytes

    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    peak, peak_src = _peaks()
    n_mean = n_prof   # particles per launch in the per-kernel leg
    # dominant kernel: the arranger (pass B).  Algorithmic bytes per particle: both passes read
    # x, v, pid, species (37 B; the cell index is cell_of(x) and is neither stored nor fetched), pass B writes the
    # same 37 B to the sorted position: 37 + 74 = 111 B per particle-step
    a_bpp, b_bpp = 37, 74
    b_bytes = b_bpp * n_mean
    b_ms = prof["pass_b"] / max(psteps, 1)
    a_bytes = a_bpp * n_mean
    a_ms = prof["pass_a"] / max(psteps, 1)
    step_bytes = a_bytes + b_bytes
    kernels = {k: round(v / max(psteps, 1), 4) for k, v in prof.items()}
    line = {
        "metric": METRIC, "value": units_all / (ms_max * 1e-3), "unit": "particle-steps/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wname, "particles": n0, "cells": w.nc, "species": len(w.species),
                   "launch": "two-step CUDA graphs replayed on the compute stream", "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "l2": "inputs larger than L2 (no flush)" if n0 * STATE_BYTES > 126e6 else
                   "state fits L2: launch-latency bound, no HBM roofline claimed"},
        "e2e": {"value": e2e_units / (e2e_ms_max * 1e-3), "unit": "particle-steps/s",
                "h2d_bytes_per_step": h2d_bytes / args.steps, "d2h_bytes_per_step": d2h_bytes / args.steps,
                "what": "bit1_load_particles(host arrays) + bit1_step(K) + bit1_get_rho(host), wall clock"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "k_pass_b (arranger: recompute push, stable scatter, fused deposit)",
                     "achieved": b_bytes / (b_ms * 1e-3) / 1e9 if b_ms > 0 else None, "peak": peak, "unit": "GB/s",
                     "frac": (b_bytes / (b_ms * 1e-3) / 1e9 / peak) if b_ms > 0 else None,
                     "traffic": _traffic("k_pass_b", args), "peak_source": peak_src,
                     "measured_in": f"a second leg of {int(psteps)} steps right after the timed region, same state, direct "
                                    "launches with CUDA events around every kernel on the compute stream (the timed "
                                    "region itself replays two-step CUDA graphs and has no per-kernel events)",
                     "bytes_per_particle": b_bpp,
                     "pass_a": {"achieved": a_bytes / (a_ms * 1e-3) / 1e9 if a_ms > 0 else None,
                                "bytes_per_particle": a_bytes / n_mean, "traffic": _traffic("k_pass_a", args)},
                     "step": {"bytes_per_particle_step": step_bytes / n_mean,
                              "achieved": step_bytes / (ms_max / args.steps * 1e-3) / 1e9,
                              "frac_of_measured_peak": step_bytes / (ms_max / args.steps * 1e-3) / 1e9 / peak,
                              "frac_of_8TBps_nominal": step_bytes / (ms_max / args.steps * 1e-3) / 1e9 / 8000.0,
                              "min_traffic_82B_equiv_GBps": 82 * n_mean / (ms_max / args.steps * 1e-3) / 1e9},
                     "kernel_ms_per_step": kernels},
        "state": {"n_live": n_end, "births": mom["births"], "far_movers_per_step": mom["far_movers"] / max(mom["step"], 1),
                  "flags": mom["flags"]},
    }
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(args)
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
