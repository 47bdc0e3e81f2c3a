"""Pins for the oracle's NEXT-2 function: wall recycling, PAPER.md:95 ("Plasma is absorbed at the walls
(depositing charge), recycling D+ ions into D neutrals"); reading N2-a."""
import numpy as np
import pytest
from scipy.special import ndtri

from helpers import py_draw
from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W

E_CH, M_E, M_DP, M_D = W.E_CHARGE, W.M_E, W.M_DP, W.M_D


def _ion_and_neutral(src_mode, vth_w=1.2e3):
    return [W.Species("i", +E_CH, M_DP, 1e10, src_mode=src_mode, src_vth=3e4, recycle_to=1, recycle_vth=vth_w),
            W.Species("n", 0.0, M_D, 1e10)]


@pytest.mark.parametrize("side", [0, 1])
@pytest.mark.parametrize("src_mode", [W.SRC_NONE, W.SRC_SELF])
def test_absorbed_ion_leaves_a_neutral_replayed_from_its_own_philox_stream(side, src_mode):
    """Brute force on one particle: position, direction and speed of the neutral from slot 14 of the parent's stream."""
    vth_w = 1.2e3
    nc, dx = 64, 1e-3
    L = nc * dx
    x0, v0 = (0.2e-3, -1e9) if side == 0 else (63.9e-3, 1e9)
    w = W.make_custom(nc, dx, 1, 1e-11, _ion_and_neutral(src_mode, vth_w), capacity=16, seed=0x1234567890ABCDEF,
                      x=[x0, 30e-3], vx=[v0, 0.0], vy=[0, 0], vz=[0, 0], sp=[0, 0])
    o = O.Oracle(w)
    o.set_E(np.zeros(nc + 1))
    o.set_step(7)
    o.step(1, freeze_field=True)
    p = o.particles()
    wc, wq = o.wall()
    assert wc[side][0] == 1 and o.recycled == 1 and o.diag()["births"] == 1
    assert o.n == (2 if src_mode == W.SRC_NONE else 3)           # the parent's own fate is unchanged
    k = p["pid"].tolist().index(2)                               # the birth takes the next pid
    assert p["sp"][k] == 1
    wd = py_draw(w.seed, 0, 7, 14)
    z = [ndtri((wd[j] + 0.5) / 2**32) for j in range(3)]
    if side == 0:
        assert p["x"][k] == 0.0 and p["cell"][k] == 0 and p["vx"][k] > 0.0
    else:
        assert p["x"][k] == L - dx * 2.0**-20 and p["x"][k] < L and p["cell"][k] == nc - 1 and p["vx"][k] < 0.0
    assert abs(p["vx"][k]) == pytest.approx(vth_w * abs(z[0]), abs=vth_w * 1e-5)
    assert p["vy"][k] == pytest.approx(vth_w * z[1], abs=vth_w * 1e-5)
    assert p["vz"][k] == pytest.approx(vth_w * z[2], abs=vth_w * 1e-5)


def test_no_recycling_without_the_setting_and_none_for_other_species():
    sp = _ion_and_neutral(W.SRC_NONE)
    sp[0].recycle_to = -1
    w = W.make_custom(64, 1e-3, 1, 1e-11, sp, capacity=16, x=[0.2e-3, 63.9e-3], vx=[-1e9, 1e9], vy=[0, 0], vz=[0, 0],
                      sp=[0, 1])
    o = O.Oracle(w)
    o.set_E(np.zeros(65))
    o.step(1, freeze_field=True)
    assert o.n == 0 and o.recycled == 0 and o.diag()["births"] == 0


def test_every_absorbed_ion_becomes_one_inward_moving_neutral_and_charge_bookkeeping_holds():
    """Config 2 with the pair source (sheath forms) and recycling: neutrals born == ions absorbed, all heading into
    the plasma when born, half-Maxwellian speeds, neutrals carry no charge (rho bookkeeping unchanged)."""
    w = W.make_config(2, scale=1 / 32, pair_source=True, recycle=True)
    o = O.Oracle(w)
    Q = o.Q()
    born_vx, born_side = [], []
    seen = set()
    for _ in range(120):
        o.step(1)
        p = o.particles()
        new = [(i, pid) for i, pid in enumerate(p["pid"].tolist()) if p["sp"][i] == 2 and pid not in seen]
        for i, pid in new:
            seen.add(pid)
            born_vx.append(p["vx"][i])
            born_side.append(0 if p["cell"][i] == 0 else 1)
            assert p["cell"][i] in (0, w.nc - 1)
    wc, wq = o.wall()
    assert o.recycled == int(wc[0][1] + wc[1][1]) == len(seen) > 20
    born_vx, born_side = np.array(born_vx), np.array(born_side)
    assert np.all(born_vx[born_side == 0] > 0) and np.all(born_vx[born_side == 1] < 0)
    # |vx| of a half-Maxwellian: mean sqrt(2/pi) vth
    vth = w.species[1].recycle_vth
    m = np.abs(born_vx).mean()
    assert abs(m - np.sqrt(2 / np.pi) * vth) < 4 * vth * np.sqrt((1 - 2 / np.pi) / len(born_vx))
    # exact charge bookkeeping: rho + wall charge - (charge injected by the pair source) is constant
    p = o.particles()
    n_e, n_i = int((p["sp"] == 0).sum()), int((p["sp"] == 1).sum())
    assert int(o.rho().sum()) == -int(Q[0]) * n_e + int(Q[1]) * n_i
    assert np.array_equal(o.dens()[2].sum(), int(Q[2]) * int((p["sp"] == 2).sum()))


# ---- second half of NEXT-2: the neutral particles' own density is the collision target (reading N2-b) ----------------

AREA = 1e-10   # m^2: brings 1e9 real particles per macro-particle to 1e19 m^-3 while Q = e*weight*2^40 = 176 stays in range


def _beam_in_neutrals(per_cell, E_eV=50.0, n_e_per_cell=400, nc=64, dt=1e-9):
    """Electrons (elastic only, all at E_eV along +y so that they stay in their cells) in a periodic box whose cell c
    holds per_cell[c] motionless neutrals at the cell centre: the target density of cell c is exactly
    per_cell-averaged-over-its-two-nodes * weight / (area dx)."""
    import math
    dx, wgt = 1.0, 1e9
    per_cell = np.asarray(per_cell)
    v = math.sqrt(2 * E_eV * E_CH / M_E)
    xe = np.repeat(np.arange(nc) + 0.5, n_e_per_cell)
    xn = np.repeat(np.arange(nc) + 0.5, per_cell)
    ne, nn = xe.shape[0], xn.shape[0]
    n_max = per_cell.max() * wgt / (AREA * dx)
    sp = [W.Species("e", -E_CH, M_E, wgt, flags=W.ELASTIC), W.Species("n", 0.0, M_D, wgt)]
    w = W.make_custom(nc, dx, 0, dt, sp, capacity=ne + nn + 16, n0=n_max, seed=77, area=AREA,
                      x=np.concatenate([xe, xn]), vx=np.zeros(ne + nn), vy=np.concatenate([np.full(ne, v), np.zeros(nn)]),
                      vz=np.zeros(ne + nn), sp=np.concatenate([np.zeros(ne, np.uint8), np.ones(nn, np.uint8)]))
    w.target_species = 1
    return w, v, n_max


def test_uniform_neutral_particles_reproduce_the_analytic_rate():
    nc, k = 64, 5
    w, v, n_max = _beam_in_neutrals(np.full(nc, k))
    o = O.Oracle(w)
    o.set_E(np.zeros(nc + 1))
    o.step(1, freeze_field=True)
    d = o.diag()
    s = w.species[0]
    n_e = int((w.sp == 0).sum())
    p = s.pnull * (n_max * 1e-19 * v) / s.numax       # every cell sits at n_max: nodes hold Q*k, their mean is k
    ev = int(d["events"][0][0])
    assert ev > 300 and abs(ev - n_e * p) <= 4.0 * np.sqrt(n_e * p * (1 - p)) + 1
    assert d["nu_overflow"] == 0
    # same box, analytic background at the same density: the same particles collide (identical random streams)
    w.target_species = -1
    o2 = O.Oracle(w)
    o2.set_E(np.zeros(nc + 1))
    o2.step(1, freeze_field=True)
    assert int(o2.diag()["events"][0][0]) == ev


def test_event_rate_follows_the_local_neutral_density_and_vanishes_where_there_are_no_neutrals():
    nc = 64
    per = np.zeros(nc, np.int64)
    per[8:24] = 2          # region A
    per[40:56] = 6         # region B: three times denser
    w, v, n_max = _beam_in_neutrals(per)
    o = O.Oracle(w)
    o.set_E(np.zeros(nc + 1))
    before = o.particles()
    o.step(1, freeze_field=True)
    after = o.particles()
    # an elastic event turns the velocity: find the electrons whose vy changed, by pid
    b = {int(p): (c, vy) for p, c, vy, s in zip(before["pid"], before["cell"], before["vy"], before["sp"]) if s == 0}
    hit_cells = [b[int(p)][0] for p, vy, s in zip(after["pid"], after["vy"], after["sp"]) if s == 0 and vy != b[int(p)][1]]
    hits = np.bincount(hit_cells, minlength=nc)
    assert hits.sum() == int(o.diag()["events"][0][0]) > 100
    interior_a, interior_b = slice(9, 23), slice(41, 55)   # cells whose two nodes both sit inside the region
    s = w.species[0]
    n_e_cell = 400
    for sl, k in ((interior_a, 2), (interior_b, 6)):
        n = hits[sl].shape[0] * n_e_cell
        p = s.pnull * ((k * 1e9 / AREA) * 1e-19 * v) / s.numax
        assert abs(hits[sl].sum() - n * p) <= 4.0 * np.sqrt(n * p * (1 - p)) + 1
    # no neutrals on either node of the cell: no events at all
    empty = np.r_[0:7, 25:39, 57:64]
    assert hits[empty].sum() == 0
    # edge cells see the mean of their two nodes (half the region's density)
    n = 2 * n_e_cell
    p = s.pnull * ((3.0 * 1e9 / AREA) * 1e-19 * v) / s.numax
    assert abs(hits[39] + hits[56] - n * p) <= 4.0 * np.sqrt(n * p * (1 - p)) + 1
