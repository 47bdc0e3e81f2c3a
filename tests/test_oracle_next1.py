"""Pins for the oracle's NEXT-1 functions: density smoothing and time-averaged
diagnostics (Table 2 `datfile` / `mvflag` / `mvStep`); readings N1-a, N1-b."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W

EPS0 = W.EPS0


def _scatter_matrix(nc, bc):
    """4 x the smoothing operator written the other way round from the oracle's gather loop: column i says
    where node i's charge goes (1 to i-1, 2 to i, 1 to i+1; a quarter leaving through a wall stays on it)."""
    ng = nc + 1 if bc else nc
    M = np.zeros((ng, ng), dtype=object)
    for i in range(ng):
        M[i, i] += 2
        for d in (-1, 1):
            j = i + d
            if bc:
                j = min(max(j, 0), ng - 1)     # folded back onto the wall node
            else:
                j %= ng
            M[j, i] += 1
    return M


@pytest.mark.parametrize("bc", [0, 1])
def test_smooth121_equals_the_scatter_form_and_conserves_charge(bc):
    rng = np.random.default_rng(11 + bc)
    for nc in (2, 3, 8, 61):
        ng = nc + 1 if bc else nc
        rho = rng.integers(-10**12, 10**12, size=ng)
        out = O.smooth121(nc, bc, rho)
        ref = _scatter_matrix(nc, bc).dot(rho.astype(object))
        assert out.tolist() == ref.tolist()
        assert int(out.astype(object).sum()) == 4 * int(rho.astype(object).sum())
    const = np.full(ng, 12345, np.int64)
    assert O.smooth121(nc, bc, const).tolist() == (4 * const).tolist()   # a uniform density is a fixed point


def test_smooth121_attenuates_a_fourier_mode_by_cos_squared():
    nc = 256
    j = np.arange(nc)
    for mode in (1, 5, 64, 127):
        k = 2 * np.pi * mode / nc
        rho = np.rint(1e9 * np.cos(k * j + 0.3)).astype(np.int64)
        out = O.smooth121(nc, 0, rho)
        want = 4.0 * np.cos(k / 2) ** 2 * 1e9 * np.cos(k * j + 0.3)
        assert np.max(np.abs(out - want)) <= 2.0 + 1e-3   # rounding of the integer input only: 4 x 0.5
    # the Nyquist mode is removed exactly
    nyq = (1 - 2 * (j % 2)) * 10**9
    assert not O.smooth121(nc, 0, nyq).any()


@pytest.mark.parametrize("cfg,passes", [(1, 1), (2, 1), (2, 3)])
def test_field_with_smoothing_is_the_poisson_solve_of_the_smoothed_charge(cfg, passes):
    w = W.make_config(cfg, scale=1 / 16)
    o = O.Oracle(w)
    o.step(3)   # config 1 loads every ion on its electron: rho == 0 until the particles move
    phi0, E0 = o.phi(), o.E()
    o.set_smoothing(passes)
    o.phase_field()
    rho = o.rho().astype(object)
    M = _scatter_matrix(w.nc, w.bc)
    for _ in range(passes):
        rho = M.dot(rho)
    assert o.rho_smoothed().tolist() == rho.tolist()
    cst = o.constants()
    Kphi, KE = cst["Kphi"], cst["KE"]
    s = 0.25 ** passes
    phi, E = O.poisson(w.nc, w.bc, Kphi * s, KE * s, np.array(rho.tolist(), np.int64))
    assert np.array_equal(phi, o.phi()) and np.array_equal(E, o.E())
    assert not np.array_equal(phi, phi0)
    if w.bc:
        # global Gauss law is untouched by the (charge-conserving) filter: E_nc - E_0 = total charge / (area eps0)
        tot = float(int(o.rho().astype(object).sum())) * 2.0**-40 / (w.area * EPS0)
        assert abs((o.E()[-1] - o.E()[0]) - tot) <= 1e-12 * max(abs(tot), np.abs(o.E()).max())
        assert abs((E0[-1] - E0[0]) - tot) <= 1e-12 * max(abs(tot), np.abs(E0).max())
    # the filter damps the grid-scale noise of the field: neighbour-to-neighbour jumps of E shrink
    assert np.abs(np.diff(o.E()[1:-1], 2)).mean() < 0.7 * np.abs(np.diff(E0[1:-1], 2)).mean()


@pytest.mark.parametrize("window,interval", [(3, 5), (1, 4), (4, 4)])
def test_time_average_is_the_sum_of_the_last_window_of_every_interval(window, interval):
    w = W.make_config(3, scale=1 / 512, n0_scale=200.0)
    o = O.Oracle(w)
    o.set_averaging(window, interval)
    dens, phi = {}, {}
    d, f, cnt, st = o.average()
    assert cnt == 0 and st == 0 and not d.any()
    for k in range(1, 3 * interval + 2):
        o.step(1)
        dens[k], phi[k] = o.dens().astype(object), o.phi()
        d, f, cnt, st = o.average()
        last = (k // interval) * interval        # the latest completed interval
        if last == 0:
            assert cnt == 0 and st == 0
            continue
        steps = range(last - window + 1, last + 1)
        assert (cnt, st) == (window, last)
        assert d.tolist() == sum(dens[i] for i in steps).tolist()
        acc = np.zeros(w.nc + 1)
        for i in steps:                          # fp64 sums in step order
            acc = acc + phi[i]
        assert np.array_equal(f, acc)
    # re-arming clears everything
    o.set_averaging(window, interval)
    assert o.average()[2] == 0
