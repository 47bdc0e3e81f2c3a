"""Pins for deposit and the integer-scan Poisson solve (SURVEY 8(c) "D", "P", "Pins")."""
from fractions import Fraction

import numpy as np
import pytest
from scipy.linalg import solve_banded

from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W

E_CH, EPS0 = W.E_CHARGE, W.EPS0


def test_deposit_single_particle_is_cic_to_fixed_point_resolution():
    sp = [W.Species("e", -E_CH, W.M_E, 1.3e11)]
    rng = np.random.default_rng(5)
    for bc in (0, 1):
        for x in list(rng.random(20) * 16.0) + [0.0, 15.999999999, 3.0, 7.5]:
            w = W.make_custom(16, 1.0, bc, 1e-12, sp, capacity=4, x=[x], vx=[0], vy=[0], vz=[0], sp=[0])
            o = O.Oracle(w)
            Q = int(o.Q()[0])
            assert Q == round(E_CH * 1.3e11 * 2**40)
            d = o.dens()[0].astype(object)
            assert sum(d) == Q and all(v >= 0 for v in d)  # exact conservation, non-negative
            c = int(x)
            j1 = (c + 1) % 16 if bc == 0 else c + 1
            assert all(v == 0 for j, v in enumerate(d) if j not in (c, j1))
            # centre of charge = x to the resolution of the 32-bit fraction and of 1/Q rounding
            frac = Fraction(int(d[j1]), Q)
            assert abs(frac - (Fraction(x) - c)) <= Fraction(1, 2**32) + Fraction(1, 2 * Q)
            assert o.rho().tolist() == (-o.dens()[0]).tolist()


def test_deposit_total_charge_and_shuffle_invariance():
    w = W.make_config(3, scale=1 / 200)
    o = O.Oracle(w)
    Q = o.Q()
    n_e = int((w.sp == 0).sum())
    n_i = int((w.sp == 1).sum())
    assert int(o.rho().sum()) == -int(Q[0]) * n_e + int(Q[1]) * n_i
    assert o.dens().sum(1).tolist() == [int(Q[0]) * n_e, int(Q[1]) * n_i]
    perm = np.random.default_rng(0).permutation(w.n)
    o2 = O.Oracle(w, load=False)
    o2.load(w.x[perm], w.vx[perm], w.vy[perm], w.vz[perm], w.sp[perm])
    assert np.array_equal(o.dens(), o2.dens()) and np.array_equal(o.rho(), o2.rho())
    # brute force per node with exact integers (python ints / Fractions)
    inv_dx = 1.0 / w.dx
    ref = [[0] * (w.nc + 1) for _ in range(2)]
    for xi, si in zip(w.x.tolist(), w.sp.tolist()):
        c = min(int(xi * inv_dx), w.nc - 1)
        f = xi * inv_dx - c
        F = min(int(Fraction(f) * 2**32), 2**32 - 1) if f > 0 else 0
        a = (int(Q[si]) * F + 2**31) >> 32
        ref[si][c] += int(Q[si]) - a
        ref[si][c + 1] += a
    assert o.dens().tolist() == ref


def _consts(nc, dx, area, bc):
    Kphi = (2.0**-40 * dx) / ((area * EPS0) * nc)
    KE = 2.0**-40 / (((2.0 * nc) * area) * EPS0)
    if not bc:
        Kphi, KE = Kphi / nc, KE / nc
    return Kphi, KE


def test_oracle_constants_match_documented_expressions():
    w = W.make_config(2, scale=1 / 64)
    o = O.Oracle(w, load=False)
    c = o.constants()
    Kphi, KE = _consts(w.nc, w.dx, w.area, 1)
    assert c["Kphi"] == Kphi and c["KE"] == KE and c["inv_dx"] == 1.0 / w.dx and c["L"] == w.nc * w.dx
    for k, s in enumerate(w.species):
        h = 0.5 * ((s.q / s.m) * w.dt)
        assert c["h"][k] == h
        t = np.array([h * b for b in w.B])
        np.testing.assert_array_equal(c["t"][k], t)
        tt = (t[0] * t[0] + t[1] * t[1]) + t[2] * t[2]
        np.testing.assert_array_equal(c["s"][k], (2.0 * t) / (1.0 + tt))


def test_poisson_bounded_matches_tridiagonal_solve_and_gauss():
    nc, dx, area = 200, 1.7e-5, 1.0
    Kphi, KE = _consts(nc, dx, area, 1)
    rng = np.random.default_rng(7)
    rho = rng.integers(-5_000_000, 5_000_000, nc + 1)
    phi, E = O.poisson(nc, 1, Kphi, KE, rho)
    kap = 2.0**-40 * dx / (area * EPS0)
    # library tridiagonal solve of phi_{j-1} - 2 phi_j + phi_{j+1} = -kap R_j, phi_0 = phi_nc = 0
    ab = np.zeros((3, nc - 1))
    ab[0, 1:] = 1.0
    ab[1, :] = -2.0
    ab[2, :-1] = 1.0
    ref = solve_banded((1, 1), ab, -kap * rho[1:nc].astype(float))
    assert phi[0] == 0.0 and phi[nc] == 0.0
    np.testing.assert_allclose(phi[1:nc], ref, rtol=0, atol=1e-11 * np.abs(ref).max())
    # interior E = centred difference of phi
    # (the difference cancels: its rounding error is ~ eps * max|phi| / dx)
    np.testing.assert_allclose(E[1:nc], -(phi[2:] - phi[:-2]) / (2 * dx), rtol=0,
                               atol=8 * np.finfo(float).eps * np.abs(phi).max() / dx)
    # global Gauss law, exact in the integers: E_nc - E_0 = 2^-40 sum(R) / (area eps0)
    num = (E[nc] - E[0]) / KE
    assert num == pytest.approx(2.0 * nc * float(rho.sum()), rel=1e-12)
    # wall-node half cells: E_{1/2} - E_0 = rho_0 (dx/2) / eps0 with all of R_0 in the half cell
    E_half = -(phi[1] - phi[0]) / dx
    tol = 8 * np.finfo(float).eps * np.abs(phi).max() / dx
    assert E_half - E[0] == pytest.approx(2.0**-40 * rho[0] / (area * EPS0), abs=tol)
    E_half_r = -(phi[nc] - phi[nc - 1]) / dx
    assert E[nc] - E_half_r == pytest.approx(2.0**-40 * rho[nc] / (area * EPS0), abs=tol)


def test_poisson_bounded_uniform_rho_is_the_parabola():
    nc, dx, area = 128, 1e-5, 1.0
    Kphi, KE = _consts(nc, dx, area, 1)
    R = 123456
    rho = np.full(nc + 1, R)
    phi, E = O.poisson(nc, 1, Kphi, KE, rho)
    rho_si = R * 2.0**-40 / (area * dx)
    x = np.arange(nc + 1) * dx
    L = nc * dx
    np.testing.assert_allclose(phi, rho_si * x * (L - x) / (2 * EPS0), rtol=1e-12, atol=1e-25)
    np.testing.assert_allclose(E[1:nc], rho_si * (x[1:nc] - L / 2) / EPS0, rtol=1e-11, atol=1e-12 * abs(E).max())


def test_poisson_bounded_single_charge_green_function():
    nc, dx, area = 64, 1e-5, 1.0
    Kphi, KE = _consts(nc, dx, area, 1)
    k = 20
    rho = np.zeros(nc + 1, np.int64)
    rho[k] = 10**9
    phi, E = O.poisson(nc, 1, Kphi, KE, rho)
    sig = 1e9 * 2.0**-40 / area  # C/m^2 sheet
    x = np.arange(nc + 1) * dx
    L, xk = nc * dx, k * dx
    g = np.where(x <= xk, x * (L - xk), xk * (L - x)) * sig / (EPS0 * L)
    np.testing.assert_allclose(phi, g, rtol=1e-12, atol=1e-30)
    assert np.argmax(phi) == k


def test_poisson_periodic_matches_fft_and_is_translation_invariant():
    nc, dx, area = 256, 1.2e-5, 1.0
    Kphi, KE = _consts(nc, dx, area, 0)
    rng = np.random.default_rng(11)
    rho = rng.integers(-10**7, 10**7, nc)
    phi, E = O.poisson(nc, 0, Kphi, KE, rho)
    assert phi[nc] == phi[0] and E[nc] == E[0] and phi[0] == 0.0
    r = (rho - rho.mean()) * 2.0**-40 / (area * dx)  # neutralising background
    rk = np.fft.fft(r)
    k = np.arange(nc)
    K2 = (2 * np.sin(np.pi * k / nc) / dx) ** 2
    pk = np.zeros_like(rk)
    pk[1:] = rk[1:] / (EPS0 * K2[1:])
    ref = np.fft.ifft(pk).real
    ref -= ref[0]  # gauge phi_0 = 0
    np.testing.assert_allclose(phi[:nc], ref, rtol=0, atol=1e-10 * np.abs(ref).max())
    Eref = -(np.roll(ref, -1) - np.roll(ref, 1)) / (2 * dx)
    np.testing.assert_allclose(E[:nc], Eref, rtol=0, atol=1e-9 * np.abs(Eref).max())
    # shifting rho shifts E exactly (integers) and phi up to the gauge constant
    phi2, E2 = O.poisson(nc, 0, Kphi, KE, np.roll(rho, 5))
    assert np.array_equal(np.roll(E[:nc], 5), E2[:nc])
    # single Fourier mode: phi_k = rho_k / (eps0 (2 sin(k dx/2)/dx)^2)
    m = 3
    amp = 10**8
    rho1 = np.round(amp * np.cos(2 * np.pi * m * np.arange(nc) / nc)).astype(np.int64)
    phi1, _ = O.poisson(nc, 0, Kphi, KE, rho1)
    a_rho = 2 * np.fft.fft(rho1 * 2.0**-40 / (area * dx))[m].real / nc
    a_phi = 2 * np.fft.fft(phi1[:nc])[m].real / nc
    assert a_phi == pytest.approx(a_rho / (EPS0 * K2[m]), rel=1e-9)


def test_poisson_exact_rational_residual_large_values():
    # magnitudes of config 5: nc = 2^20 would need seconds; use 4096 cells with huge charges so that
    # T needs more than 64 bits, and check the stencil in exact rationals.
    nc, dx, area = 4096, 5e-6, 1.0
    Kphi, KE = _consts(nc, dx, area, 1)
    rng = np.random.default_rng(13)
    rho = rng.integers(0, 2**52, nc + 1)  # one-signed: S ~ 2^64, T ~ 2^75
    phi, E = O.poisson(nc, 1, Kphi, KE, rho)
    S = [0] * (nc + 1)
    T = [0] * (nc + 1)
    for j in range(1, nc + 1):
        S[j] = S[j - 1] + int(rho[j])
        T[j] = T[j - 1] + S[j - 1]
    assert abs(T[nc]) > 2**70 and abs(S[nc]) > 2**62
    for j in (1, 2, 1000, nc // 2, nc - 1):
        exact = Fraction(Kphi) * (j * T[nc] - nc * T[j])
        assert abs(Fraction(phi[j]) - exact) <= abs(exact) * Fraction(3, 2**52)
        exactE = Fraction(KE) * (nc * (S[j - 1] + S[j]) - 2 * T[nc])
        assert abs(Fraction(E[j]) - exactE) <= abs(exactE) * Fraction(3, 2**52)
