"""The BASELINE.json workloads run to their full length at full size (opt-in, BIT1_FULL_RUNS=1: several minutes of CPU
oracle time).  Configs 1-3: every element of the final state against the oracle (SURVEY.md section 4 "100-step on configs
1-3 in full"; config 2 over its whole 1000 steps, config 3 over 300 of its 1000 by default and over all of them with
BIT1_FULL_C3_STEPS=1000, five minutes of oracle time).  Config 4: its whole 500 steps, flags
clean, exact invariants at the end.  The run made for this round is recorded in profiles/r2_full_runs.md."""
import json
import os
import time

import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import assert_state_equal, assert_moments_close

pytestmark = pytest.mark.gpu
FULL = os.environ.get("BIT1_FULL_RUNS") == "1"
REPORT = {}


def _save():
    out = os.environ.get("BIT1_REPORT_DIR")   # where to leave the figures; nothing is written without it
    if not out:
        return
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, "full_runs.json"), "w") as f:
        json.dump(REPORT, f, indent=1)


@pytest.mark.skipif(not FULL, reason="set BIT1_FULL_RUNS=1")
@pytest.mark.parametrize("cfg,steps", [(1, 100), (2, 1000), (3, int(os.environ.get("BIT1_FULL_C3_STEPS", "300")))])
def test_full_size_full_length_state_equals_oracle(cfg, steps):
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    w = W.make_config(cfg)
    g = Bit1(w)
    g.load()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(g.compute_stream)
    g.step(steps)
    ev1.record(g.compute_stream)
    g.sync()
    gpu_s = ev0.elapsed_time(ev1) * 1e-3
    o = Oracle(w)
    t0 = time.time()
    o.step(steps)
    cpu_s = time.time() - t0
    exact = assert_state_equal(g, o, where=f"config {cfg}, {steps} steps at full size")
    assert_moments_close(g, o, tol=1e-9)
    m = g.get_moments()
    REPORT[f"c{cfg}"] = dict(particles=w.n, cells=w.nc, steps=steps, gpu_s=gpu_s, oracle_s=cpu_s, bit_identical_fp64=exact,
                             births=m["births"], reinject=m["reinject"], far_movers=m["far_movers"], flags=m["flags"],
                             n_final=m["n_live"])
    _save()
    g.close()


@pytest.mark.skipif(not FULL, reason="set BIT1_FULL_RUNS=1")
def test_config4_runs_its_500_steps():
    import torch
    from paper_2606_28534_b200.binding import Bit1
    from test_gpu_fullsize import _check_invariants

    w = W.make_config(4)
    g = Bit1(w)
    g.load()
    n0 = w.n
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(g.compute_stream)
    g.step(500)
    ev1.record(g.compute_stream)
    g.sync()          # raises on any sticky flag
    gpu_s = ev0.elapsed_time(ev1) * 1e-3
    m = g.get_moments()
    assert m["step"] == 500 and m["flags"] == 0
    _check_invariants(w, g.get_particles(), g.get_rho(), g.get_dens(), m, n0 + m["births"], "step 500")
    REPORT["c4"] = dict(particles=n0, cells=w.nc, steps=500, gpu_s=gpu_s, particle_steps_per_s=n0 * 500 / gpu_s,
                        births=m["births"], reinject=m["reinject"], far_movers=m["far_movers"],
                        max_far_movers_per_step=m["max_far_movers_per_step"], flags=m["flags"], n_final=m["n_live"],
                        kinetic_J=m["kinetic_J"].tolist(), field_J=m["field_J"])
    _save()
    g.close()

