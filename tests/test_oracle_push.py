"""Pins for gather + Boris + move + boundaries (SURVEY 8(c) "G,B,M,W", "Pins")."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W
from helpers import py_draw

E_CH, M_E, M_DP = W.E_CHARGE, W.M_E, W.M_DP


def one_species(q=-E_CH, m=M_E, **kw):
    return [W.Species("e", q, m, 1e10, **kw)]


def single(x, v, *, nc=64, dx=1e-3, bc=0, dt=1e-11, B=(0, 0, 0), species=None, cap=16, **kw):
    sp = species or one_species()
    x = np.atleast_1d(np.asarray(x, float))
    v = np.atleast_2d(np.asarray(v, float))
    w = W.make_custom(nc, dx, bc, dt, sp, B=B, capacity=cap, x=x, vx=v[:, 0], vy=v[:, 1], vz=v[:, 2],
                      sp=np.zeros(x.shape[0], np.uint8), **kw)
    return O.Oracle(w), w


def test_boris_pure_B_rotation_angle_and_norm():
    # electron, B = 2 T along z, dt = 1.7726e-12 s: Omega*dt = 0.6235 (configs 2-4)
    Bz = 2.0
    Om = E_CH * Bz / M_E
    dt = 1.7726e-12
    v0 = np.array([3.0e5, -1.0e5, 2.0e5])
    # large cells so the particle stays in the periodic box; E = 0 (single species -> neutralised)
    o, w = single([0.5], [v0], nc=8, dx=1.0, dt=dt, B=(0, 0, Bz))
    o.set_E(np.zeros(9))
    expect = 2.0 * math.atan(0.5 * Om * dt)  # closed form, rotation per step
    assert expect == pytest.approx(0.6044365011758, rel=1e-12)
    phase_prev = math.atan2(v0[1], v0[0])
    total = 0.0
    nsteps = 200
    for n in range(nsteps):
        o.step(1, freeze_field=True)
        p = o.particles()
        v = np.array([p["vx"][0], p["vy"][0], p["vz"][0]])
        ph = math.atan2(v[1], v[0])
        d = (ph - phase_prev + math.pi) % (2 * math.pi) - math.pi
        # electron (q<0) gyrates counter-clockwise about +z: dphi = +angle
        assert d == pytest.approx(expect, abs=1e-13)
        total += d
        phase_prev = ph
        assert abs(np.linalg.norm(v) - np.linalg.norm(v0)) <= 4 * nsteps * np.spacing(np.linalg.norm(v0))
        assert v[2] == v0[2]
    assert total == pytest.approx(nsteps * expect, rel=1e-12)


def test_boris_oblique_B_conserves_parallel_velocity_and_speed():
    ang = math.radians(2.0)
    B = (2.0 * math.cos(ang), 2.0 * math.sin(ang), 0.0)
    b = np.array(B) / 2.0
    v0 = np.array([1.0e6, 2.0e6, -1.5e6])
    o, w = single([4.0], [v0], nc=8, dx=1.0, dt=1.7726e-12, B=B)
    o.set_E(np.zeros(9))
    o.step(50, freeze_field=True)
    p = o.particles()
    v = np.array([p["vx"][0], p["vy"][0], p["vz"][0]])
    assert np.dot(v, b) == pytest.approx(np.dot(v0, b), rel=1e-13)
    assert np.linalg.norm(v) == pytest.approx(np.linalg.norm(v0), rel=1e-13)
    # perpendicular part rotated by 50 * 2 atan(Omega dt / 2) about b (left-handed for q<0)
    th = 50 * 2.0 * math.atan(0.5 * E_CH * 2.0 / M_E * 1.7726e-12)
    vpar = np.dot(v0, b) * b
    vperp = v0 - vpar
    rot = vperp * math.cos(th) + np.cross(b, vperp) * math.sin(th)  # +th about b for q<0
    np.testing.assert_allclose(v, vpar + rot, rtol=0, atol=1e-6 * np.linalg.norm(v0))


def test_exb_drift():
    # E along x (uniform), B along z: guiding centre drifts with E x B / B^2 = (0, -E/B, 0)
    Ex, Bz = 1.0e4, 2.0
    dt = 1.7726e-12
    o, w = single([4.0], [[0.0, 0.0, 0.0]], nc=8, dx=1.0, dt=dt, B=(0, 0, Bz))
    o.set_E(np.full(9, Ex))
    th = 2.0 * math.atan(0.5 * E_CH * Bz / M_E * dt)
    nper = 2000
    nsteps = int(round(nper * 2 * math.pi / th))
    vs = np.zeros((nsteps, 3))
    for n in range(nsteps):
        o.step(1, freeze_field=True)
        p = o.particles()
        vs[n] = p["vx"][0], p["vy"][0], p["vz"][0]
    mean = vs.mean(0)
    assert mean[1] == pytest.approx(-Ex / Bz, rel=2e-3)
    assert abs(mean[0]) < 2e-3 * Ex / Bz and mean[2] == 0.0


def test_pure_E_kick_and_leapfrog_parabola():
    # exactly representable: (q/m) E dt = 2^k steps so that v_n is exact
    q, m = 1.0, 1.0
    sp = [W.Species("t", q, m, 6.0e6)]  # weight such that Q = llrint(e*w*2^40) is in range
    dt, Ex = 0.25, 0.5
    o, w = single([1.0], [[0.125, 3.0, -2.0]], nc=64, dx=1.0, dt=dt, species=sp)
    o.set_E(np.full(65, Ex))
    x, v = 1.0, 0.125
    for n in range(1, 40):
        o.step(1, freeze_field=True)
        v = v + q / m * Ex * dt
        x = x + v * dt
        p = o.particles()
        assert p["vx"][0] == v and p["vy"][0] == 3.0 and p["vz"][0] == -2.0
        assert p["x"][0] == x
        assert p["cell"][0] == int(x)


def test_linear_gather_of_E():
    # E varies linearly inside a cell: the kick uses E at the particle, dv = (q/m) E(x) dt
    q, m = 1.0, 1.0
    sp = [W.Species("t", q, m, 6.0e6)]
    E = np.arange(9, dtype=float) * 2.0  # E_j = 2 j  ->  E(x) = 2 x / dx
    for xp in (0.25, 3.5, 6.75):
        o, w = single([xp], [[0.0, 0.0, 0.0]], nc=8, dx=1.0, dt=0.125, species=sp)
        o.set_E(E)
        o.step(1, freeze_field=True)
        assert o.particles()["vx"][0] == 2.0 * xp * 0.125


def test_periodic_wrap_and_ties():
    sp = [W.Species("n", 0.0, 1.0, 6.0e6)]  # neutral: ballistic
    L = 8.0
    o, w = single([0.5, 7.5, 7.0, 0.25], [[-1, 0, 0], [1, 0, 0], [1, 0, 0], [-0.25, 0, 0]], nc=8, dx=1.0,
                  dt=1.0, species=sp)
    o.step(1, freeze_field=True)
    p = o.particles()
    got = dict(zip(p["pid"].tolist(), zip(p["x"].tolist(), p["cell"].tolist())))
    assert got[0] == (7.5, 7)   # -0.5 -> L - 0.5
    assert got[1] == (0.5, 0)   # 8.5 -> 0.5
    assert got[2] == (0.0, 0)   # x' == L is a wrap to 0 (reading A20)
    assert got[3] == (0.0, 0)
    assert o.flagword == 0


def test_absorbing_walls_count_charge_and_kill():
    sp = [W.Species("e", -E_CH, M_E, 1e10), W.Species("i", +E_CH, M_DP, 1e10)]
    x = [0.5e-3, 63.5e-3, 30e-3, 0.5e-3]
    v = [[-1e9, 0, 0], [1e9, 0, 0], [0, 0, 0], [-1e9, 0, 0]]
    w = W.make_custom(64, 1e-3, 1, 1e-11, sp, capacity=16, x=x, vx=[a[0] for a in v], vy=[0] * 4, vz=[0] * 4,
                      sp=[0, 1, 0, 1])
    o = O.Oracle(w)
    o.set_E(np.zeros(65))
    Q = o.Q()
    o.step(1, freeze_field=True)
    cnt, chg = o.wall()
    assert cnt.tolist() == [[1, 1], [0, 1]]
    assert chg.tolist() == [int(-Q[0] + Q[1]), int(Q[1])]
    p = o.particles()
    assert o.n == 1 and p["pid"].tolist() == [2]
    assert o.rho().sum() == -Q[0]


def test_reinjection_replays_the_particles_own_philox_stream():
    vth = 1.0e5
    sp = [W.Species("e", -E_CH, M_E, 1e10, src_mode=W.SRC_SELF, src_vth=vth)]
    w = W.make_custom(64, 1e-3, 1, 1e-11, sp, capacity=16, seed=0xABCDEF0123456789, x=[0.2e-3, 40e-3],
                      vx=[-1e9, 0.0], vy=[0, 0], vz=[0, 0], sp=[0, 0])
    o = O.Oracle(w)
    o.set_E(np.zeros(65))
    o.set_step(2**32 + 5)  # exercises the high word of the step counter
    o.step(1, freeze_field=True)
    p = o.particles()
    i = p["pid"].tolist().index(0)
    wd = py_draw(w.seed, 0, 2**32 + 5, 2)
    u0 = (wd[0] + 0.5) / 2**32
    xe = w.src_lo + u0 * (w.src_hi - w.src_lo)
    assert p["x"][i] == pytest.approx(xe, rel=1e-15)
    assert w.src_lo <= p["x"][i] < w.src_hi
    from scipy.special import ndtri
    for k, comp in enumerate(("vx", "vy", "vz")):
        z = ndtri((wd[1 + k] + 0.5) / 2**32)
        assert p[comp][i] == pytest.approx(vth * z, abs=vth * 1e-5)
    assert o.n == 2 and o.diag()["reinject"] == 1


def test_pair_source_births_partner_with_next_pid():
    sp = [W.Species("e", -E_CH, M_E, 1e10, flags=W.ELECTRON_PRODUCT, src_mode=W.SRC_NONE, src_vth=2e6),
          W.Species("i", +E_CH, M_DP, 1e10, flags=W.ION_PRODUCT, src_mode=W.SRC_PAIR, src_partner=0, src_vth=3e4)]
    w = W.make_custom(64, 1e-3, 1, 1e-11, sp, capacity=16, x=[0.2e-3, 40e-3, 63.9e-3], vx=[-1e9, 0.0, 1e9],
                      vy=[0] * 3, vz=[0] * 3, sp=[1, 0, 0])
    o = O.Oracle(w)
    o.set_E(np.zeros(65))
    o.step(1, freeze_field=True)
    p = o.particles()
    # ion 0 re-injected + new electron pid 3; electron pid 2 absorbed for good
    assert sorted(p["pid"].tolist()) == [0, 1, 3]
    i_ion = p["pid"].tolist().index(0)
    i_new = p["pid"].tolist().index(3)
    assert p["sp"][i_new] == 0 and p["x"][i_new] == p["x"][i_ion] and p["cell"][i_new] == p["cell"][i_ion]
    assert o.next_pid == 4 and o.diag()["births"] == 1
    # canonical order inside the cell: existing particle first, birth last
    assert i_new > i_ion
