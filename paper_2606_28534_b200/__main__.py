"""Run one of the BASELINE.json workloads through libbit1 from the command line.

    python -m paper_2606_28534_b200 --config 2 --last-step 1000 --pair-source --recycle \
        --mvflag 100 --mvstep 500 --dmpstep 500 --dump /tmp/bit1.ckpt
    python -m paper_2606_28534_b200 --config 2 --last-step 2000 --pair-source --recycle --restart /tmp/bit1.ckpt

The options follow the paper's input-deck parameters (Table 2): `Last_step`, `dmpstep` (checkpoint
interval), `mvflag` / `mvStep` (time-averaged diagnostics).  Everything runs in the library's kernels; this file only
marshals arguments and prints what the getters return.
"""
from __future__ import annotations

import argparse
import json
import os
import time


def plan_stops(step: int, last: int, dmpstep: int = 0, report: int = 0, mvstep: int = 0):
    """The step counts at which the run has to come back to the host: the multiples of every interval that lie in
    (step, last], and `last` itself.  Sorted, each once."""
    stops = {last} if last > step else set()
    for every in (dmpstep, report, mvstep):
        if every > 0:
            stops.update(range((step // every + 1) * every, last + 1, every))
    return sorted(s for s in stops if s > step)


def write_atomic(path: str, data) -> None:
    """Write the checkpoint next to `path` and rename it over it: a crash in mid-write leaves the previous file."""
    tmp = path + ".part"
    with open(tmp, "wb") as f:
        f.write(memoryview(data))
        f.flush()
        os.fsync(f.fileno())
    os.replace(tmp, path)


def main():
    ap = argparse.ArgumentParser(prog="python -m paper_2606_28534_b200")
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--scale", type=float, default=1.0, help="shrink particles and cells together")
    ap.add_argument("--last-step", type=int, default=None, help="final step (default: the workload's own length)")
    ap.add_argument("--pair-source", action="store_true", help="electrons die at the walls, lost ions return with an electron")
    ap.add_argument("--recycle", action="store_true", help="absorbed D+ ions leave D neutrals at the wall")
    ap.add_argument("--neutral-target", action="store_true", help="collide against the neutral particles' own density")
    ap.add_argument("--smooth", type=int, default=0, help="1-2-1 smoothing passes over rho")
    ap.add_argument("--mvflag", type=int, default=0, help="averaging window in steps")
    ap.add_argument("--mvstep", type=int, default=0, help="interval between averaged outputs")
    ap.add_argument("--dmpstep", type=int, default=0, help="checkpoint every this many steps")
    ap.add_argument("--dump", default=None, help="file the latest checkpoint blob is written to")
    ap.add_argument("--restart", default=None, help="checkpoint file to continue from")
    ap.add_argument("--report", type=int, default=0, help="print the moments every this many steps")
    args = ap.parse_args()

    import numpy as np
    import torch

    from . import workloads as W
    from .binding import Bit1

    w = W.make_config(args.config, scale=args.scale, pair_source=args.pair_source, recycle=args.recycle,
                      particles=args.restart is None)
    if args.neutral_target:
        if len(w.species) < 3:
            raise SystemExit("--neutral-target needs a neutral species (configs 4-5, or --recycle)")
        w.target_species = 2
    last = args.last_step if args.last_step is not None else w.steps
    sim = Bit1(w, checkpoint_staging=args.dmpstep > 0)
    sim.set_smoothing(args.smooth)
    if args.mvflag > 0:
        sim.set_averaging(args.mvflag, max(args.mvstep, args.mvflag))
    blob = torch.empty(sim.checkpoint_size(), dtype=torch.uint8).pin_memory() if args.dmpstep > 0 else None
    if args.restart:
        sim.restart(torch.from_numpy(np.fromfile(args.restart, dtype=np.uint8)))
    else:
        sim.load()
    step = sim.get_moments()["step"]
    t0 = time.perf_counter()
    units = 0
    pending = 0   # bytes of a checkpoint whose copy to the host is still in flight

    def finish_checkpoint():
        nonlocal pending
        if pending:
            sim.checkpoint_wait()
            if args.dump:
                write_atomic(args.dump, blob.numpy()[:pending])
            pending = 0

    for stop in plan_stops(step, last, args.dmpstep, args.report, args.mvstep if args.mvflag > 0 else 0):
        n_before = sim.n_live()
        sim.step(stop - step)               # enqueued; returns at once
        units += n_before * (stop - step)
        step = stop
        finish_checkpoint()                 # the previous snapshot lands and goes to disk while these steps run
        if args.dmpstep > 0 and step % args.dmpstep == 0:
            pending = sim.checkpoint(blob)  # snapshot on the device now, copy out behind the steps that follow
        if args.report > 0 and step % args.report == 0 or step == last:
            m = sim.get_moments()
            print(json.dumps({"step": m["step"], "n_live": m["n_live"], "count": m["count"].tolist(),
                              "kinetic_J": m["kinetic_J"].tolist(), "field_J": m["field_J"],
                              "wall_count": m["wall_count"].tolist(), "births": m["births"],
                              "recycled": m["recycled"], "general_steps": m["general_steps"], "flags": m["flags"]}))
        if args.mvflag > 0 and args.mvstep > 0 and step % args.mvstep == 0:
            d, f, cnt, at = sim.get_average()
            if cnt:
                print(json.dumps({"average_over_steps": cnt, "latched_at": at, "phi_mid_V": float(f[len(f) // 2] / cnt),
                                  "mean_deposit_per_species": (d.sum(axis=1) / cnt).tolist()}))
    finish_checkpoint()
    sim.sync(check_flags=False)
    dt = time.perf_counter() - t0
    print(json.dumps({"workload": w.name, "steps_run": step, "wall_s": dt,
                      "particle_steps_per_s": units / dt if dt > 0 else None}))
    sim.close()


if __name__ == "__main__":
    main()
