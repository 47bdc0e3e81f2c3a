"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Sizes span several tiles (2048 particles) and a ragged tail."""
import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import run_pair, assert_state_equal, assert_moments_close

pytestmark = pytest.mark.gpu


MODES = {"default": {}, "direct": dict(direct_launch=True), "general": dict(side_list_capacity=16, window_radius=0)}


def small(cfg, scale, **kw):
    w = W.make_config(cfg, scale=scale, **kw)
    return w


def test_load_state_matches_oracle():
    w = small(2, 1 / 64)
    g, o = run_pair(w, 0)
    assert assert_state_equal(g, o, where="load")


@pytest.mark.parametrize("mode", ["default", "direct", "general"])
@pytest.mark.parametrize("cfg,scale,kw", [
    (1, 1 / 16, {}),
    (2, 1 / 64, {}),
    (2, 1 / 64, dict(pair_source=True)),
    (3, 1 / 256, dict(n0_scale=300.0)),
    (3, 1 / 256, dict(n0_scale=300.0, pair_source=True)),
    (4, 1 / 4096, dict(n0_scale=300.0)),
    (5, 1 / 16384, dict(n0_scale=300.0)),
])
def test_one_step_state_matches_oracle(cfg, scale, kw, mode):
    """default: the fast path; direct: without CUDA graphs; general: a side list of 16 entries, so that steps with
    more far movers and births than that stall and are taken by the general path (same bits)."""
    w = small(cfg, scale, **kw)
    g, o = run_pair(w, 1, **MODES[mode])
    exact = assert_state_equal(g, o, where=f"c{cfg} 1 step")
    assert exact, "fp64 state is within tolerance but not bit-identical"


@pytest.mark.parametrize("mode", ["default", "general"])
@pytest.mark.parametrize("cfg,scale,kw,steps", [
    (1, 1.0, {}, 100),
    (2, 1 / 16, {}, 100),
    (2, 1 / 16, dict(pair_source=True), 100),
    (3, 1 / 64, dict(n0_scale=100.0), 100),
    (4, 1 / 1024, dict(n0_scale=100.0), 100),
    (5, 1 / 4096, dict(n0_scale=100.0), 100),
])
def test_hundred_steps_match_oracle(cfg, scale, kw, steps, mode):
    w = small(cfg, scale, **kw)
    g, o = run_pair(w, steps, **MODES[mode])
    assert_state_equal(g, o, where=f"c{cfg} {steps} steps")
    assert_moments_close(g, o, tol=1e-9)


@pytest.mark.parametrize("cfg,scale,kw", [
    (4, 1 / 16, dict(n0_scale=30.0)),     # 1.25e7 particles, 4096 cells: 4 CTAs in the cooperative kernels, 41 tiles per CTA
    (5, 1 / 64, dict(n0_scale=30.0)),     # 1.56e7 particles, 16384 cells: 16 CTAs in k_mid and k_field
])
def test_mid_size_state_matches_oracle_element_by_element(cfg, scale, kw):
    """Large enough that the persistent passes reload their stages dozens of times and the cooperative kernels (cell
    scan, column scan, field solve) run on several CTAs, small enough for the oracle: every element compared."""
    w = small(cfg, scale, **kw)
    g, o = run_pair(w, 3)
    exact = assert_state_equal(g, o, where=f"c{cfg} x{scale:g}, 3 steps")
    assert exact, "fp64 state, phi and E are within tolerance but not bit-identical"
    g.close()
