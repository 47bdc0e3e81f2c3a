"""GPU parity for SURVEY 8(f) NEXT-1: density smoothing and time-averaged diagnostics
(PAPER.md:79-83), through the C ABI against the CPU oracle; readings N1-a, N1-b."""
import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import assert_state_equal

pytestmark = pytest.mark.gpu


def _pair(w, passes=0, window=0, interval=0, **kw):
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    g = Bit1(w, **kw)
    g.set_smoothing(passes)
    g.set_averaging(window, interval)
    g.load()
    o = Oracle(w, load=False)
    o.set_smoothing(passes)
    o.set_averaging(window, interval)
    o.load(w.x, w.vx, w.vy, w.vz, w.sp)
    return g, o


@pytest.mark.parametrize("cfg,scale,kw,passes", [
    (1, 1 / 4, {}, 1),
    (2, 1 / 16, dict(pair_source=True), 1),
    (3, 1 / 64, dict(n0_scale=100.0), 2),
    (5, 1 / 4096, dict(n0_scale=100.0), 8),
])
def test_smoothed_field_matches_oracle_bit_for_bit(cfg, scale, kw, passes):
    w = W.make_config(cfg, scale=scale, **kw)
    g, o = _pair(w, passes=passes)
    assert np.array_equal(g.get_rho_smoothed(), o.rho_smoothed()), "load: smoothed rho"
    assert assert_state_equal(g, o, where=f"c{cfg} smoothing load")
    g.step(30)
    o.step(30)
    g.sync(check_flags=False)
    assert np.array_equal(g.get_rho_smoothed(), o.rho_smoothed()), "smoothed rho"
    assert assert_state_equal(g, o, where=f"c{cfg} smoothing x{passes}, 30 steps")
    # switching it off again takes effect at the next step
    g.set_smoothing(0)
    o.set_smoothing(0)
    g.step(3)
    o.step(3)
    g.sync(check_flags=False)
    assert assert_state_equal(g, o, where=f"c{cfg} smoothing off again")
    g.close()


@pytest.mark.parametrize("window,interval", [(3, 5), (1, 4), (4, 4)])
def test_time_averages_match_oracle_bit_for_bit(window, interval):
    w = W.make_config(3, scale=1 / 128, n0_scale=100.0)
    g, o = _pair(w, passes=1, window=window, interval=interval)
    assert g.get_average()[2:] == (0, 0)
    done = 0
    for chunk in (2, 3, 1, 7, 4, 6):   # bit1_step(n) with averaging armed, in uneven chunks
        g.step(chunk)
        o.step(chunk)
        done += chunk
        dg, fg, cg, sg = g.get_average()
        do, fo, co, so = o.average()
        assert (cg, sg) == (co, so) == ((window, (done // interval) * interval) if done >= interval else (0, 0))
        assert np.array_equal(dg, do) and np.array_equal(fg, fo), f"after {done} steps"
    assert assert_state_equal(g, o, where="averaging run")
    g.close()


@pytest.mark.parametrize("staging", [False, True])
def test_restart_carries_settings_and_running_sums(staging):
    import torch
    from paper_2606_28534_b200.binding import Bit1

    w = W.make_config(3, scale=1 / 128, n0_scale=100.0)
    g, o = _pair(w, passes=2, window=4, interval=6, checkpoint_staging=staging)
    g.step(9)   # mid-window: steps 9 of window 9..12 already accumulated
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    g.checkpoint(blob)
    g.step(2)
    g.checkpoint_wait()
    g.close()
    h = Bit1(w, checkpoint_staging=staging)   # settings come from the blob
    h.restart(blob)
    h.step(6)
    o.step(15)
    h.sync(check_flags=False)
    dg, fg, cg, sg = h.get_average()
    do, fo, co, so = o.average()
    assert (cg, sg) == (co, so) == (4, 12)
    assert np.array_equal(dg, do) and np.array_equal(fg, fo)
    assert np.array_equal(h.get_rho_smoothed(), o.rho_smoothed())
    assert assert_state_equal(h, o, where="restart with NEXT-1 state")
    h.close()


def test_argument_checks():
    from paper_2606_28534_b200 import binding as B

    w = W.make_config(1, scale=1 / 16)
    g = B.Bit1(w)
    for bad in (-1, 9):
        with pytest.raises(B.Bit1Error):
            g.set_smoothing(bad)
    with pytest.raises(B.Bit1Error):
        g.set_averaging(5, 3)
    with pytest.raises(B.Bit1Error):
        g.set_averaging(-1, 3)
    g.set_averaging(0, 0)
    g.close()
