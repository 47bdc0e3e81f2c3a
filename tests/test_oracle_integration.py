"""Whole-step pins for the oracle (SURVEY 8(c) "Pins": cold-plasma oscillation, energy drift,
charge bookkeeping, restart, sheath)."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W

E_CH, M_E, M_DP, EPS0 = W.E_CHARGE, W.M_E, W.M_DP, W.EPS0


def test_cold_plasma_oscillation_frequency():
    # cold electrons on a fixed neutralising background (periodic mode subtracts the mean charge),
    # mode-1 displacement << dx: field energy ~ cos^2(w t), w = (2/dt) asin(wpe dt / 2) (leapfrog).
    n_ref, nc, ppc = 1e18, 256, 64
    wpe = math.sqrt(n_ref * E_CH**2 / (EPS0 * M_E))
    lam = math.sqrt(EPS0 * 10.0 / (n_ref * E_CH))
    dx, dt = 0.5 * lam, 0.1 / wpe
    L = nc * dx
    N = nc * ppc
    x0 = (np.arange(N) + 0.5) * (L / N)
    amp = 1e-3 * dx
    x = (x0 + amp * np.sin(2 * np.pi * x0 / L)) % L
    sp = [W.Species("e", -E_CH, M_E, n_ref * L / N)]
    w = W.make_custom(nc, dx, 0, dt, sp, capacity=N + 8, x=x, vx=np.zeros(N), vy=np.zeros(N), vz=np.zeros(N),
                      sp=np.zeros(N, np.uint8))
    o = O.Oracle(w)
    nsteps = 700
    k1 = np.exp(-2j * np.pi * np.arange(nc) / nc)
    a = np.zeros(nsteps + 1)
    a[0] = (o.E()[:nc] * k1).sum().imag  # xi ~ sin(kx) -> E ~ sin(kx)
    for n in range(nsteps):
        o.step(1)
        a[n + 1] = (o.E()[:nc] * k1).sum().imag
    # mode amplitude ~ cos(w t): zero crossings by linear interpolation
    idx = np.flatnonzero(np.sign(a[:-1]) != np.sign(a[1:]))
    tz = idx + a[idx] / (a[idx] - a[idx + 1])
    assert tz.shape[0] >= 20  # > 10 periods
    half_period = (tz[-1] - tz[0]) / (tz.shape[0] - 1)
    omega = math.pi / (half_period * dt)
    expect = (2.0 / dt) * math.asin(0.5 * wpe * dt)
    assert expect / wpe == pytest.approx(1.000417, abs=2e-6)
    assert omega == pytest.approx(expect, rel=1e-3)
    assert abs(omega / wpe - 1.0) < 2e-3
    assert o.rho().sum() == -int(o.Q()[0]) * N


def test_config1_energy_drift_and_exact_neutrality():
    w = W.make_config(1)
    o = O.Oracle(w)
    assert np.all(o.rho() == 0)  # ions loaded on top of electrons
    m0 = o.moments()
    tot0 = m0["kinetic_J"].sum() + m0["field_J"]
    worst = 0.0
    for _ in range(10):
        o.step(10)
        assert int(o.rho().sum()) == 0
        m = o.moments()
        worst = max(worst, abs(m["kinetic_J"].sum() + m["field_J"] - tot0) / tot0)
    assert worst < 1e-4  # SURVEY 8(c) pins: <= 2.4e-5 seen in the prototype
    assert o.n == w.n and o.flagword == 0
    assert m["field_J"] / m["kinetic_J"].sum() < 5e-3


def test_restart_reproduces_the_uninterrupted_run_bit_for_bit():
    w = W.make_config(3, scale=1 / 200, n0_scale=100.0)
    a = O.Oracle(w)
    a.step(12)
    snap = a.snapshot()
    a.step(9)
    b = O.Oracle(w, load=False)
    b.restore(snap)
    b.step(9)
    pa, pb = a.particles(), b.particles()
    for k in pa:
        assert np.array_equal(pa[k], pb[k]), k
    assert np.array_equal(a.rho(), b.rho()) and np.array_equal(a.E(), b.E()) and np.array_equal(a.phi(), b.phi())
    assert a.next_pid == b.next_pid and a.step_index == b.step_index == 21
    assert np.array_equal(a.wall()[0], b.wall()[0]) and np.array_equal(a.wall()[1], b.wall()[1])


def test_charge_bookkeeping_with_walls_and_sources():
    # literal SRC_SELF: every absorbed particle comes back -> sum(rho) never changes, N constant
    w = W.make_config(2, scale=1 / 32)
    o = O.Oracle(w)
    tot0 = int(o.rho().sum())
    o.step(40)
    cnt, chg = o.wall()
    Q = o.Q()
    assert cnt.sum() > 0 and o.n == w.n and int(o.rho().sum()) == tot0
    assert int(chg.sum()) == int((cnt.astype(np.int64) * (np.array([-1, 1]) * Q)[None, :]).sum())
    # pair source: electrons die at the walls, every lost ion returns with a new electron
    w = W.make_config(2, scale=1 / 32, pair_source=True)
    o = O.Oracle(w)
    tot0 = int(o.rho().sum())
    o.step(60)
    cnt, chg = o.wall()
    births = o.diag()["births"]
    assert cnt[:, 0].sum() > 0
    # rho + wall charge - injected charge is constant: absorbed e (-Q_e each) removed, ion re-injection
    # puts +Q_i back and adds a born electron (-Q_e)
    inj = int(cnt[:, 1].sum()) * int(Q[1]) - births * int(Q[0])
    assert int(o.rho().sum()) + int(chg.sum()) - inj == tot0
    assert o.n == w.n - int(cnt[:, 0].sum()) + births
    assert chg[0] < 0 and chg[1] < 0  # electrons reach the walls first (PAPER.md:95 sheath)


def test_sheath_forms_with_pair_source():
    # plasma absorbed at the walls, a sheath forms.  Pair-source variant (reading A9),
    # cut down to 512 cells.  The sudden start rings the bulk at wpe (+-300 V, 62.8 steps per period);
    # averaged over two plasma periods the bulk potential sits at the floating-wall estimate
    # Te*[0.5 ln((m_D/(2 pi m_e))/(1+Ti/Te)) + 0.5..0.7] = 3.3-3.6 Te (SURVEY 8(c) pins; accept 2.8-4.5 Te),
    # and the wall field points into both walls.
    w = W.make_config(2, scale=1 / 8, pair_source=True)
    o = O.Oracle(w)
    o.step(378)
    acc = []
    for _ in range(126):
        o.step(1)
        acc.append(o.phi()[w.nc // 4: 3 * w.nc // 4].mean())
    Te = 20.0
    bulk = float(np.mean(acc))
    assert 2.8 * Te < bulk < 4.5 * Te
    E = o.E()
    assert E[0] < 0 < E[w.nc]
    cnt, chg = o.wall()
    assert cnt[:, 0].sum() > 4 * cnt[:, 1].sum() and chg[0] < 0 and chg[1] < 0
