"""Randomised parity: seeded random combinations of workload, size, collision rate, sources, recycling, neutral target,
smoothing, averaging, window radius (adaptive or pinned) and its bound, side-list capacity (small ones force the general
path), launch mode, velocity scale and step chunking, CUDA path vs oracle, every element compared, no case skipped.
BIT1_FUZZ_CASES (default 24) sets how many cases run; BIT1_FUZZ_SEED shifts the sequence; BIT1_FUZZ_BIG=1 draws 4e5 to
2.5e6 particles per case instead of 7e2 to 7e4."""
import os

import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import assert_state_equal

pytestmark = pytest.mark.gpu

N_CASES = int(os.environ.get("BIT1_FUZZ_CASES", "24"))
SEED0 = int(os.environ.get("BIT1_FUZZ_SEED", "0"))


def _case(seed):
    rng = np.random.default_rng(1000003 * SEED0 + seed)
    cfg = int(rng.integers(1, 6))
    full_n = {1: 204800, 2: 1638400, 3: 1e7, 4: 2e8, 5: 1e9}[cfg]
    sizes = [700, 3000, 9000, 30000, 70000]
    if os.environ.get("BIT1_FUZZ_BIG") == "1":       # several tiles per CTA: the stages are reloaded, cooperative grids > 1
        sizes = [400000, 900000, 2500000]
    n_target = float(rng.choice(sizes))
    thin = float(rng.choice([1.0, 1.0, 0.25, 0.04]))     # keep this fraction: fewer particles per cell, more cells
    kw = dict(scale=n_target / full_n / thin)
    if cfg >= 3:
        kw["n0_scale"] = float(rng.choice([1.0, 100.0, 1000.0, 5000.0]))
    if cfg >= 2:
        kw["pair_source"] = bool(rng.integers(0, 2))
        kw["recycle"] = bool(rng.integers(0, 2))
    opts = dict(passes=int(rng.choice([0, 0, 1, 3])), window=0, interval=0,
                boost=float(rng.choice([1.0, 1.0, 6.0, 40.0])), R=int(rng.choice([-1, -1, 1, 0, 2, 4])),
                chunks=[int(c) for c in rng.integers(1, 14, size=int(rng.integers(1, 5)))],
                target=bool(cfg >= 4 and rng.integers(0, 2)), gen_seed=int(rng.integers(1, 2**31)),
                lib_seed=int(rng.integers(1, 2**62)), restart=bool(rng.integers(0, 3) == 0), thin=thin)
    if rng.integers(0, 2):
        opts["interval"] = int(rng.integers(1, 7))
        opts["window"] = int(rng.integers(1, opts["interval"] + 1))
    # arranger internals (none changes a result): window radius adaptive (-1) or pinned, its upper bound, the side-list
    # capacity (small ones send steps through the general path), direct launches instead of graph replay
    b1 = dict(window_radius=None if opts["R"] < 0 else opts["R"], window_radius_max=int(rng.choice([0, 0, 1, 4, 60])),
              side_list_capacity=int(rng.choice([0, 0, 0, 16, 300, 5000])), direct_launch=bool(rng.integers(0, 4) == 0),
              checkpoint_staging=bool(rng.integers(0, 2)))
    opts["bit1"] = b1
    return cfg, kw, opts


@pytest.mark.parametrize("seed", range(N_CASES))
def test_random_case_matches_oracle(seed):
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    cfg, kw, op = _case(seed)
    w = W.make_config(cfg, gen_seed=op["gen_seed"], lib_seed=op["lib_seed"], **kw)
    if op["thin"] < 1.0:
        keep = np.sort(np.random.default_rng(seed).choice(w.n, size=max(1, int(w.n * op["thin"])), replace=False))
        for k in ("x", "vx", "vy", "vz", "sp"):
            setattr(w, k, np.ascontiguousarray(getattr(w, k)[keep]))
    for k in ("vx", "vy", "vz"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k) * op["boost"]))
    if op["target"]:
        w.target_species = 2
    g = Bit1(w, **op["bit1"])
    o = Oracle(w, load=False)
    for side in (g, o):
        side.set_smoothing(op["passes"])
        side.set_averaging(op["window"], op["interval"])
    g.load()
    o.load(w.x, w.vx, w.vy, w.vz, w.sp)
    where = f"fuzz seed {seed}: c{cfg} {kw} {op}"
    for i, c in enumerate(op["chunks"]):
        g.step(c)
        o.step(c)
        if op["restart"] and i == 0:
            blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
            g.checkpoint(blob)
            g.checkpoint_wait()
            g.close()
            g = Bit1(w, **op["bit1"])
            g.restart(blob)
    g.sync(check_flags=False)
    assert assert_state_equal(g, o, where=where)   # whatever path the steps took (fast, side list, general): same bits
    dg, fg, cg, sg = g.get_average()
    do, fo, co, so = o.average()
    assert (cg, sg) == (co, so) and np.array_equal(dg, do) and np.array_equal(fg, fo), where
    g.close()
