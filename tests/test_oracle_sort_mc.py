"""Pins for the stable sort/compaction and the null-collision Monte Carlo
(SURVEY 8(c) "S", "C", "A", "Pins")."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W
from helpers import py_draw

E_CH, M_E, M_DP, M_D = W.E_CHARGE, W.M_E, W.M_DP, W.M_D


def test_sort_equals_library_stable_sort_with_deaths_and_births():
    # pair-source variant with boosted collisions: deaths (electrons at walls), births (pair + ionisation)
    w = W.make_config(3, scale=1 / 100, n0_scale=300.0, pair_source=True)
    o = O.Oracle(w)
    for _ in range(3):
        n0 = o.n
        o.phase_push()
        pre = o.particles()  # slots 0..n-1 in old order, then births; dead have cell -1
        assert o.n_slots >= n0
        keep = np.flatnonzero(pre["cell"] >= 0)
        order = keep[np.argsort(pre["cell"][keep], kind="stable")]  # library routine
        o.phase_sort()
        post = o.particles()
        for k in pre:
            assert np.array_equal(post[k], pre[k][order]), k
        cs = o.cell_start()
        assert cs[0] == 0 and cs[-1] == o.n == order.shape[0]
        assert np.array_equal(np.diff(cs), np.bincount(post["cell"], minlength=w.nc))
        assert np.all(np.diff(post["cell"]) >= 0)
        o.phase_deposit()
        o.phase_field()
        o.set_step(o.step_index + 1)
    d = o.diag()
    assert d["births"] > 20 and o.wall()[0].sum() > 0
    # pids are unique and births got consecutive ids after the loaded ones
    p = o.particles()["pid"]
    assert np.unique(p).shape[0] == p.shape[0]
    assert o.next_pid == w.n + d["births"]


def beam(n, E_eV, m, q, flags, *, n0, dt=1e-10, seed=9, extra_species=()):
    """n particles of one species moving along +x with energy E_eV; periodic, E=0, B=0."""
    v = math.sqrt(2 * E_eV * E_CH / m)
    sp = [W.Species("b", q, m, 1e9, flags=flags)] + list(extra_species)
    nc, dx = 64, 1.0
    x = (np.arange(n) + 0.5) * (nc * dx / n)
    w = W.make_custom(nc, dx, 0, dt, sp, capacity=3 * n + 16, n0=n0, seed=seed, x=x, vx=np.full(n, v),
                      vy=np.zeros(n), vz=np.zeros(n), sp=np.zeros(n, np.uint8))
    o = O.Oracle(w)
    o.set_E(np.zeros(nc + 1))
    return o, w, v


def four_sigma(k, n, p):
    return abs(k - n * p) <= 4.0 * math.sqrt(n * p * (1 - p)) + 1


def test_elastic_rate_and_energy_loss_law():
    n, E0, n0 = 400_000, 50.0, 2e20
    o, w, v = beam(n, E0, M_E, -E_CH, W.ELASTIC, n0=n0)
    s = w.species[0]
    before = o.particles()
    o.step(1, freeze_field=True)
    d = o.diag()
    p_evt = s.pnull * (n0 * 1e-19 * v) / s.numax  # exact null-collision probability (SURVEY "MC rates")
    assert p_evt == pytest.approx(n0 * 1e-19 * v * w.dt, rel=0.05)
    assert four_sigma(int(d["candidates"][0]), n, s.pnull)
    assert four_sigma(int(d["events"][0, 0]), n, p_evt)
    assert d["events"][0, 1] == 0 and d["events"][0, 2] == 0 and d["births"] == 0
    after = o.particles()
    idx = np.argsort(after["pid"])
    va = np.stack([after["vx"][idx], after["vy"][idx], after["vz"][idx]], 1)
    vb = np.stack([before["vx"], before["vy"], before["vz"]], 1)[np.argsort(before["pid"])]
    changed = np.flatnonzero(np.any(va != vb, axis=1))
    assert changed.shape[0] == d["events"][0, 0]
    g0 = np.linalg.norm(vb[changed], axis=1)
    g1 = np.linalg.norm(va[changed], axis=1)
    cosx = np.einsum("ij,ij->i", va[changed], vb[changed]) / (g0 * g1)
    ratio = (g1 / g0) ** 2
    np.testing.assert_allclose(ratio, 1 - 2 * (M_E / M_D) * (1 - cosx), rtol=1e-12)
    # isotropic scattering: cos(chi) uniform on (-1, 1)
    from scipy import stats
    assert stats.kstest(cosx, "uniform", args=(-1, 2)).pvalue > 1e-3


def test_ionisation_rate_energy_balance_and_births():
    n, E0, n0 = 300_000, 80.0, 4e22
    ion = W.Species("i", +E_CH, M_DP, 1e9, flags=W.ION_PRODUCT)
    o, w, v = beam(n, E0, M_E, -E_CH, W.IONISE | W.ELECTRON_PRODUCT, n0=n0, extra_species=(ion,))
    s = w.species[0]
    sig = 4e-18 * math.log(E0 / 13.6) / (E0 * 13.6)
    before = o.particles()
    o.step(1, freeze_field=True)
    d = o.diag()
    p_evt = s.pnull * (n0 * sig * v) / s.numax
    nev = int(d["events"][0, 1])
    assert four_sigma(nev, n, p_evt) and nev > 500
    assert d["births"] == 2 * nev and o.n == n + 2 * nev and o.next_pid == n + 2 * nev
    after = o.particles()
    by_pid = {int(p): i for i, p in enumerate(after["pid"])}
    vb = {int(p): (before["vx"][i], before["vy"][i], before["vz"][i]) for i, p in enumerate(before["pid"])}
    ev = lambda i: 0.5 * M_E * (after["vx"][i] ** 2 + after["vy"][i] ** 2 + after["vz"][i] ** 2) / E_CH
    # parents in index (= pid, here) order get births next_pid + 2r (electron), + 2r + 1 (ion)
    parents = sorted(p for p in range(n) if (after["vx"][by_pid[p]], after["vy"][by_pid[p]], after["vz"][by_pid[p]]) != vb[p])
    assert len(parents) == nev
    vi = []
    for r, p in enumerate(parents):
        ie, ii, ip = by_pid[n + 2 * r], by_pid[n + 2 * r + 1], by_pid[p]
        assert after["sp"][ie] == 0 and after["sp"][ii] == 1
        assert after["x"][ie] == after["x"][ip] == after["x"][ii]
        assert ev(ip) + ev(ie) == pytest.approx(E0 - 13.6, rel=1e-12)
        vi.append((after["vx"][ii], after["vy"][ii], after["vz"][ii]))
        # the split fraction is the SP slot of the parent's own stream
        wd = py_draw(w.seed, p, 0, 3)
        u = (((wd[0] << 32 | wd[1]) >> 12) + 0.5) / 2**52
        assert ev(ip) == pytest.approx(u * (E0 - 13.6), rel=1e-12)
    vi = np.array(vi)
    # born ions: Maxwellian at the neutral temperature (table variance 0.99996617)
    var = vi.var(0) / w.vth_n**2
    assert np.all(np.abs(var - 1.0) < 5 * math.sqrt(2.0 / nev))


def test_charge_exchange_rate_and_velocity_swap():
    n, n0 = 300_000, 2e22
    E0 = 30.0
    o, w, v = beam(n, E0, M_DP, +E_CH, W.CX | W.TARGET_MAXWELLIAN, n0=n0, dt=1e-9)
    s = w.species[0]
    o.step(1, freeze_field=True)
    d = o.diag()
    nev = int(d["events"][0, 2])
    # relative speed |v - vn| ~ v (vn << v): rate within the spread of g
    p_evt = s.pnull * (n0 * 5e-19 * v) / s.numax
    assert abs(nev - n * p_evt) < 4 * math.sqrt(n * p_evt) + 0.02 * n * p_evt
    assert four_sigma(int(d["candidates"][0]), n, s.pnull)
    after = o.particles()
    changed = np.flatnonzero(after["vx"] != v)
    assert changed.shape[0] == nev
    from scipy.special import ndtri
    for i in changed[:200]:
        wd = py_draw(w.seed, int(after["pid"][i]), 0, 1)  # slot NV
        for k, comp in enumerate(("vx", "vy", "vz")):
            z = ndtri((wd[k] + 0.5) / 2**32)
            assert after[comp][i] == pytest.approx(w.vth_n * z, abs=w.vth_n * (1e-5 if abs(z) < 3 else 5e-3))
    vs = np.stack([after["vx"][changed], after["vy"][changed], after["vz"][changed]], 1)
    assert np.all(np.abs(vs.var(0) / w.vth_n**2 - 1.0) < 5 * math.sqrt(2.0 / nev))


def test_branching_ratio_elastic_vs_ionisation():
    n, E0, n0 = 400_000, 100.0, 1e22
    ion = W.Species("i", +E_CH, M_DP, 1e9, flags=W.ION_PRODUCT)
    o, w, v = beam(n, E0, M_E, -E_CH, W.ELASTIC | W.IONISE | W.ELECTRON_PRODUCT, n0=n0, extra_species=(ion,))
    o.step(1, freeze_field=True)
    d = o.diag()
    sig_i = 4e-18 * math.log(E0 / 13.6) / (E0 * 13.6)
    n_el, n_io = int(d["events"][0, 0]), int(d["events"][0, 1])
    tot = n_el + n_io
    frac = sig_i / (sig_i + 1e-19)
    assert tot > 2000 and abs(n_io - tot * frac) < 4 * math.sqrt(tot * frac * (1 - frac))
    assert d["nu_overflow"] == 0


def test_no_collision_below_threshold_and_for_flagless_species():
    o, w, v = beam(50_000, 10.0, M_E, -E_CH, W.IONISE | W.ELECTRON_PRODUCT, n0=1e23,
                   extra_species=(W.Species("i", +E_CH, M_DP, 1e9, flags=W.ION_PRODUCT),))
    o.step(1, freeze_field=True)
    assert o.diag()["events"].sum() == 0 and o.diag()["candidates"][0] > 0
    o, w, v = beam(1000, 10.0, M_E, -E_CH, 0, n0=1e23)
    o.step(1, freeze_field=True)
    assert o.diag()["candidates"].sum() == 0


def test_no_ionisation_inside_the_table_interval_that_holds_the_threshold():
    """Reading R-thr: the 0.5 eV table interpolates to a positive cross-section on (13.5, 13.6] eV; an ionisation
    there would hand out E - 13.6 < 0 (NaN speeds).  The rule 'zero at or below the threshold' forbids it."""
    ion = W.Species("i", +E_CH, M_DP, 1e9, flags=W.ION_PRODUCT)
    for E_eV, expect_events in ((13.58, False), (13.6 - 1e-9, False), (13.7, True)):
        o, w, v = beam(200_000, E_eV, M_E, -E_CH, W.IONISE | W.ELECTRON_PRODUCT, n0=3e24, extra_species=(ion,))
        assert O.lib().orc_sigma(o.h, 1, E_eV) > 0.0          # the table alone would allow it
        o.step(1, freeze_field=True)
        d = o.diag()
        p = o.particles()
        assert d["candidates"][0] > 1000
        assert (d["events"][0][1] > 0) == expect_events and (d["births"] > 0) == expect_events
        for k in ("x", "vx", "vy", "vz"):
            assert np.all(np.isfinite(p[k]))
        assert o.flagword == 0


def test_capacity_flag():
    n, n0 = 20_000, 4e23
    ion = W.Species("i", +E_CH, M_DP, 1e9, flags=W.ION_PRODUCT)
    o, w, v = beam(n, 80.0, M_E, -E_CH, W.IONISE | W.ELECTRON_PRODUCT, n0=n0, extra_species=(ion,))
    w.capacity = n + 5
    o = O.Oracle(w)
    o.set_E(np.zeros(w.nc + 1))
    o.step(1, freeze_field=True)
    assert o.flagword & 1 and o.n == n + 5
