"""GPU parity for SURVEY 8(f) NEXT-2, wall recycling (absorbed D+ ions leave D neutrals at the wall),
through the C ABI against the CPU oracle; reading N2-a."""
import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import run_pair, assert_state_equal, assert_moments_close

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,scale,kw,steps", [
    (2, 1 / 32, dict(pair_source=True), 100),       # a neutral species that starts empty
    (2, 1 / 32, {}, 60),                             # literal re-injection of the absorbed ion + its neutral
    (3, 1 / 128, dict(n0_scale=200.0, pair_source=True), 100),   # recycled neutrals next to ionisation births
    (4, 1 / 2048, dict(n0_scale=100.0), 100),        # three loaded species
    (5, 1 / 8192, dict(n0_scale=100.0), 40),
])
def test_recycling_matches_oracle_bit_for_bit(cfg, scale, kw, steps):
    w = W.make_config(cfg, scale=scale, recycle=True, **kw)
    # hotter ions so that cut-down runs see wall hits of the recycling species within a few dozen steps
    ions = w.sp == 1
    for k in ("vx", "vy", "vz"):
        getattr(w, k)[ions] *= 30.0
    g, o = run_pair(w, steps)
    assert o.recycled > 0, "the workload was meant to recycle"
    assert assert_state_equal(g, o, where=f"c{cfg} recycling, {steps} steps")
    assert_moments_close(g, o, tol=1e-9)
    g.close()


def test_restart_with_recycling_and_rejection_without_it():
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1, Bit1Error, ERR_CHECKPOINT

    w = W.make_config(2, scale=1 / 32, pair_source=True, recycle=True)
    w.vx[w.sp == 1] *= 30.0
    g = Bit1(w)
    g.load()
    g.step(25)
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    g.checkpoint(blob)
    g.checkpoint_wait()
    g.close()
    h = Bit1(w)
    h.restart(blob)
    h.step(25)
    h.sync(check_flags=False)
    o = Oracle(w)
    o.step(50)
    assert o.recycled > 0
    assert assert_state_equal(h, o, where="restart with recycling")
    h.close()
    # the recycling setting is part of the configuration a blob is validated against
    w2 = W.make_config(2, scale=1 / 32, pair_source=True, recycle=True)
    w2.species[1].recycle_to = -1
    k = Bit1(w2)
    with pytest.raises(Bit1Error) as e:
        k.restart(blob)
    assert e.value.status == ERR_CHECKPOINT
    with pytest.raises(Bit1Error):
        k.set_recycling(1, 7, 1.0)
    with pytest.raises(Bit1Error):
        k.set_recycling(1, 2, -1.0)
    k.close()


# ---- second half of NEXT-2: neutral particles as the collision target (reading N2-b) ---------------------------------

def _boost_collisions(w, f=3000.0):
    """Cut-down runs see few events at physical rates: scale the cross-section tables by f and bound the rate for 1.5 x
    the largest neutral-particle density of the load (inputs only: the library sees tables, numax and pnull)."""
    import math
    neutrals = w.x[w.sp == 2]
    peak = np.bincount(np.minimum((neutrals / w.dx).astype(np.int64), w.nc - 1), minlength=w.nc).max()
    n_bound = 1.5 * peak * w.species[2].weight / (w.area * w.dx)
    for name in ("sig_el", "sig_ion", "sig_cx"):
        setattr(w, name, getattr(w, name) * f)
    for s in w.species:
        if s.numax > 0.0:
            s.numax = s.numax * f * n_bound / w.n0
            s.pnull = 1.0 - math.exp(-s.numax * w.dt)
    w.target_species = 2


@pytest.mark.parametrize("cfg,scale,steps", [(4, 1 / 2048, 100), (5, 1 / 8192, 60)])
def test_neutral_particle_target_matches_oracle_bit_for_bit(cfg, scale, steps):
    w = W.make_config(cfg, scale=scale, recycle=True)
    _boost_collisions(w)
    g, o = run_pair(w, steps)
    d = o.diag()
    assert d["events"].sum() > 200 and d["births"] > 20, "the workload was meant to collide"
    assert assert_state_equal(g, o, where=f"c{cfg} neutral-particle target, {steps} steps")
    assert_moments_close(g, o, tol=1e-9)
    g.close()


def test_neutral_particle_target_in_a_periodic_box_and_restart():
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1, Bit1Error, ERR_CHECKPOINT
    from test_oracle_next2 import _beam_in_neutrals

    per = np.zeros(64, np.int64)
    per[8:24] = 2
    per[40:64] = 6          # reaches the last cell: its right node is node 0 (periodic wrap)
    w, v, n_max = _beam_in_neutrals(per)
    g, o = run_pair(w, 6)
    assert o.diag()["events"].sum() > 300
    assert assert_state_equal(g, o, where="periodic box, neutral-particle target")
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    g.checkpoint(blob)
    g.checkpoint_wait()
    g.close()
    h = Bit1(w)
    h.restart(blob)
    h.step(6)
    h.sync(check_flags=False)
    o.step(6)
    assert assert_state_equal(h, o, where="restart, neutral-particle target")
    h.close()
    w.target_species = -1      # another configuration: the blob is rejected
    k = Bit1(w)
    with pytest.raises(Bit1Error) as e:
        k.restart(blob)
    assert e.value.status == ERR_CHECKPOINT
    with pytest.raises(Bit1Error):
        k.set_neutral_target(5)
    k.close()
