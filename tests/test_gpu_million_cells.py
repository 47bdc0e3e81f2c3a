"""The code paths only a grid of more than 148 x 4096 cells reaches, at a size the oracle finishes in seconds:
BASELINE.json configs[4]'s 1 048 576 cells (and a periodic box of the same size) with about 16 particles per cell
instead of 954 -- k_mid's cell scan and tile-descriptor loop run several chunks per CTA on all 148 CTAs, k_field's range
scan likewise, the cooperative grids sit at their 148-CTA cap, tiles span about 64 cells (dozens at the Gaussian
peak, hundreds at its edges, where the window overflows into the side list).  Every element is compared."""
import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import run_pair, assert_state_equal

pytestmark = pytest.mark.gpu


def test_configs4_grid_bounded_every_element_after_three_steps():
    w = W.make_config(5, ppc_scale=1 / 60, n0_scale=100.0)   # 1.67e7 particles, B = 2 T at 3 deg, walls, collisions
    assert w.nc == 1048576 and w.nc > 148 * 4096
    g, o = run_pair(w, 3)
    exact = assert_state_equal(g, o, where="1 048 576 cells, bounded")
    assert exact, "fp64 state, phi and E are within tolerance but not bit-identical"
    m = g.get_moments()
    assert m["far_movers"] > 0 and m["general_steps"] == 0
    g.close()


def test_million_cell_periodic_box_every_element_after_three_steps():
    w = W.make_config(1, scale=1024, ppc_scale=0.08)         # 1 048 576 cells, 1.68e7 particles, periodic, B = 0
    assert w.nc == 1048576 and w.bc == 0
    g, o = run_pair(w, 3)
    exact = assert_state_equal(g, o, where="1 048 576 cells, periodic")
    assert exact, "fp64 state, phi and E are within tolerance but not bit-identical"
    g.close()
