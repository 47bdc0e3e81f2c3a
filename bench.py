#!/usr/bin/env python
"""bench.py -- particle-steps/s of the PIC-MC hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--scale 1.0] [--impl reference]

One "step" is one whole timestep (mover, side-list ordering + cell scan, arranger with fused deposit, field
solve) over every particle of the workload.  Default workload: BASELINE.json configs[3] (2e8 particles, 65536
cells, exponential sheath profile, 3 species, config-3 collisions) -- the first configuration at the
"1e8+ particles" size that the metric's HBM target is quoted on; configs[4] (1e9) also fits one GPU and is timed in
the `workloads` leg from device-generated inputs (its 33 GB of host-side inputs would take minutes to make and pin).
Inputs are larger than L2 (8.2 GB state vs 126 MB), so no L2 flush is needed between steps.

Legs of one run: (1) W warm-up steps, then K timed steps bracketed by CUDA events on the compute stream (`value`;
bit1_step replays two-step CUDA graphs); (2) min(K, 50) more steps with CUDA events around every kernel (`roofline`);
(3) end to end: bit1_load_particles from pinned host arrays + K steps + bit1_get_rho to the host, wall clock (`e2e`);
(4) at N = 1, legs (1)-(2) again for the other four configurations of BASELINE.json (`workloads`; configs[4]'s 1e9
particles are generated on the device); (5) at N = 1, the CPU oracle on a bounded cut-down of the headline workload,
one core and one plain process per host core (`cpu_baseline`).

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


FULL_N = {1: 204800, 2: 1638400, 3: 1e7, 4: 2e8, 5: 1e9}
A_BPP, B_BPP = 37, 74   # algorithmic bytes per particle of pass A / pass B; 111 B per step
MIN_BPP = 82            # read the 41 B state once, write it once


def _workload(cfg: int, scale: float, rank: int, **kw):
    from paper_2606_28534_b200 import workloads as W

    w = W.make_config(cfg, scale=scale, gen_seed=2606285340 + cfg + 1000 * rank,
                      lib_seed=2606285340000 + cfg + 1000 * rank, **kw)
    name = f"BASELINE.json configs[{cfg - 1}]" + (f" cut down x{scale:g}" if scale != 1.0 else "")
    return w, name


def _oracle_worker(job):
    """One plain oracle process: a cut-down of the configuration with its own generator seed, stepped for about
    `seconds`; returns (particle-steps, seconds).  The oracle itself stays single-threaded (oracle/bit1_oracle.c)."""
    cfg, scale, seed, seconds = job
    from oracle.oracle import Oracle
    from paper_2606_28534_b200 import workloads as W

    w = W.make_config(cfg, scale=scale, gen_seed=seed)
    o = Oracle(w)
    o.step(1)
    steps = 0
    t0 = time.perf_counter()
    while True:
        o.step(2)
        steps += 2
        if time.perf_counter() - t0 > seconds or steps >= 400:
            break
    return float(w.n) * steps, time.perf_counter() - t0, w.n, w.nc, steps


def _cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(cfg: int, scale: float, seconds: float = 10.0, all_cores: bool = True):
    """The oracle as it stands on a bounded cut-down of the same configuration: (i) one process, (ii) one plain
    process per host core on disjoint cut-downs (different generator seeds), aggregate particle-steps/s."""
    import multiprocessing as mp

    target_n = 4.0e6
    sc = scale * min(1.0, target_n / (FULL_N[cfg] * scale))
    units, dt, n, nc, steps = _oracle_worker((cfg, sc, 2606285340 + cfg, seconds))
    single = units / dt
    sample = (f"configs[{cfg - 1}] cut down to {n} particles / {nc} cells (same particles per cell and profile), "
              f"gcc -O2 -ffp-contract=off, plain single-threaded oracle")
    out = {"value": single, "unit": UNIT, "cores": 1, "kind": "oracle", "cpu_model": _cpu_model(),
           "host_cores": os.cpu_count(), "sample": sample + f"; {steps} steps in {dt:.1f} s on one core"}
    ncores = os.cpu_count() or 1
    if all_cores and ncores > 1:
        ctx = mp.get_context("spawn")
        jobs = [(cfg, sc, 2606285340 + cfg + 7919 * (k + 1), seconds) for k in range(ncores)]
        t0 = time.perf_counter()
        with ctx.Pool(ncores) as pool:
            res = pool.map(_oracle_worker, jobs)
        agg = sum(r[0] / r[1] for r in res)
        out = {"value": agg, "unit": UNIT, "cores": ncores, "kind": "oracle", "cpu_model": _cpu_model(),
               "host_cores": ncores, "single_thread": single,
               "sample": sample + f"; one such process per host core ({ncores}) on disjoint cut-downs, each about "
                                  f"{seconds:.0f} s, aggregate of the processes' own rates; one core alone: {single:.3g}"}
    return out


def run_reference(args):
    rank, world, _ = _dist()
    if rank != 0:
        return
    from oracle.oracle import Oracle
    from paper_2606_28534_b200 import workloads as W

    sc = args.scale * min(1.0, 4.0e6 / (FULL_N[args.config] * args.scale))
    w = W.make_config(args.config, scale=sc)
    o = Oracle(w)
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    val = w.n * args.steps / dt
    sample = (f"each step = one oracle timestep on configs[{args.config - 1}] cut down to {w.n} particles / {w.nc} "
              f"cells; single thread ({_cpu_model()}, {os.cpu_count()} host cores)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "particle-steps/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}] (bounded sample)", "particles": w.n,
                       "cells": w.nc},
            "cpu_baseline": {"value": val, "unit": "particle-steps/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "particle-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def _measure(sim, steps: int, warmup: int, peak: float, barrier=None, sampler_index=None):
    """W warm-up steps, K timed steps (CUDA events on the compute stream), then min(K, 50) steps with events around
    every kernel.  The state must be loaded.  Returns a dict of raw figures."""
    import torch

    sim.step(warmup)
    sim.sync()
    n_start = sim.n_live()
    general0 = sim.get_moments()["general_steps"]
    launches0 = sim.launch_count()
    ev0 = torch.cuda.Event(enable_timing=True)
    ev1 = torch.cuda.Event(enable_timing=True)
    if barrier:
        barrier()
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    t_wall0 = time.perf_counter()
    with torch.cuda.stream(sim.compute_stream):
        ev0.record(sim.compute_stream)
        sim.step(steps)
        ev1.record(sim.compute_stream)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    t_wall1 = time.perf_counter()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms = ev0.elapsed_time(ev1)
    launches = sim.launch_count() - launches0
    sim.sync()
    ms_settled = 1e3 * (time.perf_counter() - t_wall0)   # wall clock incl. any step redone by the general path
    # A step whose side list overflowed is a device no-op inside the event pair; its real work (the general path) runs in
    # the sync above.  If that happened in the timed leg the event time undercounts: the wall clock up to the end of the
    # settle is the honest figure, and every number derived from `ms` (headline value, workloads list) uses it.
    general_timed = int(sim.get_moments()["general_steps"] - general0)
    ms_events = ms
    if general_timed > 0:
        ms = ms_settled
    n_end = sim.n_live()
    units = 0.5 * (n_start + n_end) * steps
    psteps_want = min(steps, 50)
    sim.profile(True)
    sim.step(psteps_want)
    prof, psteps = sim.get_profile()
    sim.profile(False)
    sim.sync()
    n_prof = 0.5 * (n_end + sim.n_live())
    mom = sim.get_moments()
    kern = {k: v / max(psteps, 1) for k, v in prof.items()}
    return dict(ms=ms, ms_events=ms_events, ms_settled=ms_settled, general_timed=general_timed,
                timed="wall clock incl. settle of redone steps" if general_timed else "CUDA events",
                units=units, launches=int(launches), clocks=clocks, n_end=n_end,
                n_prof=n_prof, kern=kern, psteps=int(psteps), mom=mom)


def _sustained(sim, steps: int, sampler_index: int):
    """What a long run gets: `steps` more steps of the loaded workload (its own length, e.g. configs[3]'s 500) in one
    bit1_step call, timed by CUDA events on the compute stream, with the clock sampler running throughout (a 20-step
    burst is over before nvidia-smi's 100 ms poll fires twice; under the power cap the SM clock, and the step time with
    it, drifts during the first seconds)."""
    import torch

    sampler = ClockSampler(sampler_index)
    time.sleep(0.3)   # the sampler's first rows
    general0 = sim.get_moments()["general_steps"]
    n_start = sim.n_live()
    ev0 = torch.cuda.Event(enable_timing=True)
    ev1 = torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    with torch.cuda.stream(sim.compute_stream):
        ev0.record(sim.compute_stream)
        sim.step(steps)
        ev1.record(sim.compute_stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    clocks = sampler.stop(t0, t1)
    ms = ev0.elapsed_time(ev1)
    sim.sync()
    ms_settled = 1e3 * (time.perf_counter() - t0)
    general = int(sim.get_moments()["general_steps"] - general0)
    if general > 0:   # redone steps ran in the sync, outside the event pair (see _measure)
        ms = ms_settled
    units = 0.5 * (n_start + sim.n_live()) * steps
    return {"steps": steps, "ms_per_step": ms / steps, "value": units / (ms * 1e-3), "unit": UNIT,
            "seconds": ms * 1e-3, "sm_mhz_median": clocks.get("sm_mhz"), "sm_max_mhz": clocks.get("sm_max_mhz"),
            "reasons": clocks.get("reasons"), "clock_samples": clocks.get("samples"),
            "general_steps": general, "timed": "wall clock incl. settle of redone steps" if general else "CUDA events"}


def _summary(r, steps: int, peak: float, n0: int):
    """Figures of one workload for the `workloads` list."""
    ms_step = r["ms"] / steps
    n = r["n_prof"]
    resident = n0 * STATE_BYTES <= 126e6
    b_ms, a_ms = r["kern"]["pass_b"], r["kern"]["pass_a"]
    out = {"value": r["units"] / (r["ms"] * 1e-3), "ms_per_step": ms_step, "steps": steps,
           "kernel_ms_per_step": {k: round(v, 4) for k, v in r["kern"].items()},
           "GBps_on_111B": (A_BPP + B_BPP) * n / (ms_step * 1e-3) / 1e9,
           "frac_on_111B": (A_BPP + B_BPP) * n / (ms_step * 1e-3) / 1e9 / peak,
           "frac_on_82B_minimum": MIN_BPP * n / (ms_step * 1e-3) / 1e9 / peak,
           "pass_b_frac": (B_BPP * n / (b_ms * 1e-3) / 1e9 / peak) if b_ms > 0 else None,
           "pass_a_frac": (A_BPP * n / (a_ms * 1e-3) / 1e9 / peak) if a_ms > 0 else None,
           "l2": "state fits L2: launch-latency bound, the fractions are not HBM roofline claims" if resident else
                 "state larger than L2 (no flush)",
           "far_movers_per_step": r["mom"]["far_movers"] / max(r["mom"]["step"], 1),
           "window_radius": r["mom"]["window_radius"], "general_steps": r["mom"]["general_steps"],
           "general_steps_in_timed_region": r["general_timed"], "timed": r["timed"],
           "flags": r["mom"]["flags"], "gpu_launches": r["launches"]}
    return out


def _side_workloads(args, local: int, peak: float):
    """The other four configurations of BASELINE.json (north_star: "throughput on the five synthetic workloads"), timed
    the same way as the headline one; configs[4] (1e9 particles) is generated on the device (workloads.device_particles)."""
    import torch

    from paper_2606_28534_b200 import workloads as W
    from paper_2606_28534_b200.binding import Bit1

    out = []
    for cfg in (1, 2, 3, 5):
        if cfg == args.config:
            continue
        entry = {"workload": f"BASELINE.json configs[{cfg - 1}]", "particles": int(FULL_N[cfg])}
        try:
            t0 = time.perf_counter()
            steps = max(args.steps, 50) if cfg <= 3 else args.steps
            if cfg == 5:
                free, total = torch.cuda.mem_get_info()
                if total < 170e9:
                    entry["skipped"] = f"needs about 150 GB of device memory, {total / 1e9:.0f} GB present"
                    out.append(entry)
                    continue
                w = W.make_config(5, particles=False)
                sim = Bit1(w, device=f"cuda:{local}")
                dev = W.device_particles(w, 5, torch.device("cuda", local))
                torch.cuda.synchronize()
                sim.load_particles(*dev)
                n0 = int(dev[0].shape[0])
                del dev
                torch.cuda.empty_cache()
                entry["data"] = "synthetic, generated on the device (same recipe as the host generator)"
            else:
                w, _ = _workload(cfg, 1.0, 0)
                sim = Bit1(w, device=f"cuda:{local}")
                sim.load()
                n0 = w.n
            entry["cells"] = int(w.nc)
            entry["setup_s"] = round(time.perf_counter() - t0, 2)
            r = _measure(sim, steps, args.warmup, peak)
            entry.update(_summary(r, steps, peak, n0))
            sim.close()
            del sim
            torch.cuda.empty_cache()
        except Exception as e:  # a side workload must never take the headline line down
            entry["error"] = f"{type(e).__name__}: {e}"
        out.append(entry)
    return out


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

    gen_kw = {}
    if args.noisy:
        gen_kw["quiet"] = False
    w, wname = _workload(args.config, args.scale, rank, **gen_kw)
    if args.vscale != 1.0:
        for k in ("vx", "vy", "vz"):
            setattr(w, k, np.ascontiguousarray(getattr(w, k) * args.vscale))
    n0 = w.n
    bit1_kw = {}
    if args.radius is not None:
        bit1_kw["window_radius"] = args.radius
    if args.radius_max:
        bit1_kw["window_radius_max"] = args.radius_max
    if args.side_list:
        bit1_kw["side_list_capacity"] = args.side_list
    sim = Bit1(w, device=f"cuda:{local}", **bit1_kw)
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

    peak, peak_src = _peaks()
    # ---- device-resident leg: W warm-up steps, then exactly K timed steps; then the per-kernel leg ------------------
    sim.load_particles(host["x"], host["vx"], host["vy"], host["vz"], host["sp"])
    r = _measure(sim, args.steps, args.warmup, peak, barrier=barrier, sampler_index=local if rank == 0 else None)
    ms, units, launches, clocks, n_end = r["ms"], r["units"], r["launches"], r["clocks"], r["n_end"]
    prof, psteps, n_prof, mom = r["kern"], r["psteps"], r["n_prof"], r["mom"]
    ms_max, units_all = aggregate(ms, units, world, dev)
    sustained = None
    if world == 1 and args.sustained_steps != 0:
        k = args.sustained_steps if args.sustained_steps > 0 else min(int(w.steps), 1000)
        sustained = _sustained(sim, k, local)

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
    n_mean = n_prof   # particles per launch in the per-kernel leg
    # dominant kernel: the arranger (pass B).  Algorithmic bytes per particle: both passes read
    # x, v, pid, species (37 B; the cell index is cell_of(x) and is neither stored nor fetched), pass B writes the
    # same 37 B to the sorted position: 37 + 74 = 111 B per particle-step
    a_bpp, b_bpp = A_BPP, B_BPP
    b_bytes = b_bpp * n_mean
    b_ms = prof["pass_b"]
    a_bytes = a_bpp * n_mean
    a_ms = prof["pass_a"]
    step_bytes = a_bytes + b_bytes
    kernels = {k: round(v, 4) for k, v in prof.items()}
    ms_step = ms_max / args.steps
    line = {
        "metric": METRIC, "value": units_all / (ms_max * 1e-3), "unit": "particle-steps/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wname, "particles": n0, "cells": w.nc, "species": len(w.species),
                   "headline": "configs[3] is the headline: the first configuration at the 1e8+ particles the metric's HBM "
                               "target is quoted on whose host-side inputs (8 GB) load in seconds; configs[4] (1e9, the "
                               "largest that fits one GPU) and configs[0..2] are under `workloads`",
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
                              "achieved": step_bytes / (ms_step * 1e-3) / 1e9,
                              "frac_of_measured_peak": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
                              "frac_of_8TBps_nominal": step_bytes / (ms_step * 1e-3) / 1e9 / 8000.0,
                              "min_traffic_82B_equiv_GBps": MIN_BPP * n_mean / (ms_step * 1e-3) / 1e9,
                              "frac_on_82B_minimum": MIN_BPP * n_mean / (ms_step * 1e-3) / 1e9 / peak},
                     "kernel_ms_per_step": kernels},
        "state": {"n_live": n_end, "births": mom["births"], "far_movers_per_step": mom["far_movers"] / max(mom["step"], 1),
                  "window_radius": mom["window_radius"], "general_steps": mom["general_steps"],
                  "general_steps_in_timed_region": r["general_timed"], "timed": r["timed"], "flags": mom["flags"]},
    }
    if sustained is not None:
        sustained["what"] = (f"{sustained['steps']} further steps of the same loaded state in one bit1_step call (the "
                             "workload's own run length), after the timed region and the per-kernel leg")
        line["sustained"] = sustained
    sim.close()
    del sim, pin, host
    torch.cuda.empty_cache()
    if world == 1 and args.workloads == "all":
        line["workloads"] = [dict(workload=wname, particles=n0, cells=int(w.nc), headline=True,
                                  **_summary(r, args.steps, peak, n0))] + _side_workloads(args, local, peak)
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(args.config, args.scale)
    print(json.dumps(line))


def run_sweep(args):
    """profiles/r2_far_mover_sweep.md: ms/step of one configuration against the fraction of particles that leave their
    tile's sort window, made by scaling the loaded velocities with the window radius pinned (the side list takes the
    far movers, the general path takes over beyond its capacity) and adaptive (the window widens instead).  Prints one
    JSON line per point."""
    import numpy as np
    import torch

    from paper_2606_28534_b200.binding import Bit1

    torch.cuda.set_device(0)
    peak, _ = _peaks()
    w, wname = _workload(args.config, args.scale, 0, quiet=not args.noisy)
    base = {k: getattr(w, k).copy() for k in ("vx", "vy", "vz")}
    for radius in (1, None):
        for vs in (1.0, 1.5, 2.0, 2.5, 3.0, 4.0, 6.0, 10.0, 40.0):
            for k in base:
                setattr(w, k, np.ascontiguousarray(base[k] * vs))
            kw = dict(window_radius_max=args.radius_max or 40)
            if radius is not None:
                kw["window_radius"] = radius
            sim = Bit1(w, device="cuda:0", **kw)
            sim.load()
            steps = args.steps
            r = _measure(sim, steps, args.warmup, peak)
            m = r["mom"]
            # steps redone by the general path run when the host next waits: their time is in the wall clock only
            ms = r["ms_settled"] if m["general_steps"] else r["ms_events"]
            print(json.dumps({"workload": wname + ("" if not args.noisy else " (independent load)"), "vscale": vs,
                              "radius": "adaptive" if radius is None else radius, "ms_per_step": round(ms / steps, 3),
                              "timed": "wall clock incl. settle" if m["general_steps"] else "CUDA events",
                              "far_mover_fraction": m["far_movers"] / max(m["step"], 1) / max(r["n_end"], 1),
                              "max_far_movers_per_step": m["max_far_movers_per_step"], "window_radius": m["window_radius"],
                              "general_steps": m["general_steps"], "steps_total": m["step"], "flags": m["flags"],
                              "kernel_ms_per_step": {k: round(v, 3) for k, v in r["kern"].items()}}), flush=True)
            sim.close()
            del sim
            torch.cuda.empty_cache()


def run_stream_overlap(args):
    """profiles/r2_stream_overlap.md: ms/step of the configuration alone, with bit1_checkpoint (staged) every K steps and
    with bit1_stream_publish every K steps while a consumer thread drains the ring; CUDA events around the whole leg."""
    import threading

    import torch

    from paper_2606_28534_b200.binding import Bit1

    torch.cuda.set_device(0)
    w, wname = _workload(args.config, args.scale, 0)
    sim = Bit1(w, device="cuda:0", checkpoint_staging=True)
    sim.load()
    sim.step(args.warmup)
    sim.sync()
    total = args.steps

    def timed(every, what):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        with torch.cuda.stream(sim.compute_stream):
            ev0.record(sim.compute_stream)
            done = 0
            while done < total:
                k = min(every or total, total - done)
                sim.step(k)
                done += k
                if every and what == "checkpoint":
                    sim.checkpoint(blob)
                elif every and what == "stream":
                    sim.stream_publish()
            ev1.record(sim.compute_stream)
        sim.sync()
        wall = time.perf_counter() - t0
        sim.checkpoint_wait()
        return ev0.elapsed_time(ev1) / total, 1e3 * wall / total

    # every leg is compared with a plain leg run right before it: under the power cap the step time drifts by a few
    # per cent over a minute of load, more than a snapshot costs
    def plain():
        ev, wall = timed(0, None)
        print(json.dumps({"workload": wname, "leg": "steps only", "steps": total, "ms_per_step_events": round(ev, 4),
                          "ms_per_step_wall": round(wall, 4)}), flush=True)
        return ev, wall

    blob = torch.empty(sim.checkpoint_size(), dtype=torch.uint8).pin_memory()
    for every in args.every:
        base_ev, base_wall = plain()
        ev, wall = timed(every, "checkpoint")
        print(json.dumps({"workload": wname, "leg": f"bit1_checkpoint (staged) every {every} steps", "steps": total,
                          "snapshot_GB": round(sim.checkpoint_size() / 1e9, 2), "ms_per_step_events": round(ev, 4),
                          "ms_per_step_wall": round(wall, 4),
                          "overhead_events_pct": round(100 * (ev / base_ev - 1), 2),
                          "overhead_wall_pct": round(100 * (wall / base_wall - 1), 2)}),
              flush=True)
    del blob
    slot = (sim.stream_slot_size() + 255) // 256 * 256
    ring = torch.empty(2 * slot, dtype=torch.uint8).pin_memory()
    sim.stream_open(ring, 2)
    seen, stop = [], threading.Event()

    def consumer():
        last = 0
        while True:
            got = sim.stream_acquire(last)
            if got is None:
                if stop.is_set():
                    return
                time.sleep(0.001)
                continue
            last, snap = got
            # a consumer in the paper's sense: per-species density profile from the counts per cell
            seen.append((snap["step"], [int(r["counts"].sum()) for r in snap["species"]]))
            sim.stream_release(last)

    t = threading.Thread(target=consumer)
    t.start()
    for every in args.every:
        base_ev, base_wall = plain()
        n_seen = len(seen)
        ev, wall = timed(every, "stream")
        print(json.dumps({"workload": wname, "leg": f"bit1_stream_publish every {every} steps + consumer thread",
                          "steps": total, "slot_GB": round(slot / 1e9, 2), "ms_per_step_events": round(ev, 4),
                          "ms_per_step_wall": round(wall, 4),
                          "overhead_events_pct": round(100 * (ev / base_ev - 1), 2),
                          "overhead_wall_pct": round(100 * (wall / base_wall - 1), 2),
                          "snapshots_consumed": len(seen) - n_seen}), flush=True)
    stop.set()
    t.join()
    sim.stream_close()
    sim.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--workloads", default="all", choices=["all", "none"],
                    help="all: also time the other four configurations (key `workloads` of the line)")
    # measurement knobs (profiles/r2_far_mover_sweep.md): none of them changes a result
    ap.add_argument("--vscale", type=float, default=1.0, help="multiply the loaded velocities (hotter plasma)")
    ap.add_argument("--noisy", action="store_true", help="load the charged species independently (no quiet start)")
    ap.add_argument("--radius", type=int, default=None, help="pin the sort-window radius (default: adaptive)")
    ap.add_argument("--radius-max", type=int, default=0)
    ap.add_argument("--side-list", type=int, default=0, help="side-list capacity (entries)")
    ap.add_argument("--sustained-steps", type=int, default=-1,
                    help="length of the `sustained` leg (default: the workload's own step count, at most 1000; 0 = skip)")
    ap.add_argument("--sweep", default=None, choices=["far-movers", "stream"],
                    help="print the far-mover sweep / the checkpoint-overlap table instead of the bench line")
    ap.add_argument("--every", type=int, nargs="+", default=[200, 100, 50], help="--sweep stream: snapshot intervals")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    if args.sweep == "stream":
        run_stream_overlap(args)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
