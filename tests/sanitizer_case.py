#!/usr/bin/env python
"""One small parity case for compute-sanitizer (SURVEY section 4 "Sanitizers", section 5 "Race detection").

    compute-sanitizer --tool {memcheck,racecheck,synccheck,initcheck} python tests/sanitizer_case.py --config 3

Loads a cut-down of the configuration, steps it (direct launches and, with --graph, CUDA-graph replays), optionally
checkpoints and restarts half way, and compares every element with the CPU oracle.  Exit code 0 = parity holds; the
sanitizer's own report is what profiles/r2_sanitizer.md records.
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--particles", type=float, default=2.0e4)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--graph", action="store_true", help="8 more steps through bit1_step's CUDA-graph path")
    ap.add_argument("--restart", action="store_true")
    ap.add_argument("--boost", type=float, default=1.0, help="velocity scale (hot variants stress the side list)")
    args = ap.parse_args()

    import numpy as np
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200 import workloads as W
    from paper_2606_28534_b200.binding import Bit1
    from parity import assert_state_equal

    full_n = {1: 204800, 2: 1638400, 3: 1e7, 4: 2e8, 5: 1e9}[args.config]
    kw = dict(scale=args.particles / full_n)
    if args.config >= 3:
        kw["n0_scale"] = 300.0
    if args.config >= 2:
        kw["pair_source"] = True
        kw["recycle"] = True
    w = W.make_config(args.config, **kw)
    for k in ("vx", "vy", "vz"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k) * args.boost))
    g = Bit1(w)
    g.load()
    o = Oracle(w)
    g.step(args.steps)
    o.step(args.steps)
    if args.restart:
        blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
        g.checkpoint(blob)
        g.checkpoint_wait()
        g.close()
        g = Bit1(w)
        g.restart(blob)
        g.step(2)
        o.step(2)
    if args.graph:
        g.step(8)
        o.step(8)
    g.sync(check_flags=False)
    exact = assert_state_equal(g, o, where="sanitizer case")
    m = g.get_moments(density=True)
    print(f"sanitizer case ok: config {args.config}, {o.n} particles, step {m['step']}, births {m['births']}, "
          f"far movers {m['far_movers']}, flags {m['flags']}, bit-identical {exact}")
    g.close()


if __name__ == "__main__":
    main()
