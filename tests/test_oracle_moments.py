"""Pins for the oracle's diagnostics: orc_get_moments and orc_get_density (SURVEY 8(c) "Moments"; PAPER.md:79-83,
Table 2: the input deck's diagnostics).  Every expected value is computed here from the definition in exact rational
arithmetic (fractions.Fraction) on hand-chosen inputs, never from the oracle's own formula: a dropped 1/2, a missing
weight or mass, a missing wall-node factor or a wrong cell volume each fail one named test below."""
from fractions import Fraction as Fr

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_28534_b200 import workloads as W

E_CH, EPS0 = W.E_CHARGE, W.EPS0


def _two_species(nc, dx, bc, x, v, sp, *, w_e=3.0e9, w_i=7.0e9, area=0.5):
    """Two species with DIFFERENT masses and weights (a swapped or missing factor shows)."""
    species = [W.Species("e", -E_CH, W.M_E, w_e), W.Species("D+", +E_CH, W.M_DP, w_i)]
    v = np.asarray(v, dtype=np.float64).reshape(-1, 3)
    return W.make_custom(nc, dx, bc, 1e-12, species, area=area, capacity=len(x) + 8, x=x, vx=v[:, 0], vy=v[:, 1],
                         vz=v[:, 2], sp=sp)


def test_kinetic_energy_and_momentum_are_half_m_w_sum_v2_and_m_w_sum_vx():
    # velocities exactly representable, so the exact rational sums are what fp64 must round to (one rounding per
    # product at most: bound 4 ulp)
    x = [0.25, 1.5, 2.75, 3.5, 0.75, 2.25, 3.25]
    v = [(3.0, -4.0, 12.0), (-1.5, 2.5, 0.5), (1024.0, 0.0, -0.125), (7.0, 7.0, 7.0),   # electrons
         (-2.0, 1.0, 2.0), (0.5, 0.25, -8.0), (100.0, -100.0, 50.0)]                    # ions
    sp = [0, 0, 0, 0, 1, 1, 1]
    w = _two_species(4, 1.0, 1, x, v, sp)
    o = O.Oracle(w)
    m = o.moments()
    assert m["count"].tolist() == [4, 3]
    for s, spc in enumerate(w.species):
        vv = [Fr(a) for (a, b, c), t in zip(v, sp) if t == s]
        v2 = sum(Fr(a) ** 2 + Fr(b) ** 2 + Fr(c) ** 2 for (a, b, c), t in zip(v, sp) if t == s)
        ke = Fr(1, 2) * Fr(spc.m) * Fr(spc.weight) * v2
        px = Fr(spc.m) * Fr(spc.weight) * sum(vv)
        assert abs(Fr(float(m["kinetic_J"][s])) - ke) <= 4 * Fr(2) ** -52 * ke, f"kinetic_J[{s}]"
        assert abs(Fr(float(m["px"][s])) - px) <= 4 * Fr(2) ** -52 * abs(px), f"px[{s}]"
    # the two species differ by mass AND weight: swapping either between them is a factor 3670 or 2.33
    assert m["kinetic_J"][0] != m["kinetic_J"][1]


def test_kinetic_energy_scales_with_weight_and_mass_separately():
    x, v, sp = [0.5, 1.5], [(2.0, 0.0, 0.0), (0.0, 3.0, 0.0)], [0, 1]
    a = O.Oracle(_two_species(4, 1.0, 0, x, v, sp, w_e=1e9, w_i=1e9)).moments()
    b = O.Oracle(_two_species(4, 1.0, 0, x, v, sp, w_e=4e9, w_i=1e9)).moments()
    assert b["kinetic_J"][0] == 4.0 * a["kinetic_J"][0] and b["kinetic_J"][1] == a["kinetic_J"][1]
    assert b["px"][0] == 4.0 * a["px"][0]
    # energy ratio between one electron and one ion at known speeds is (m_e * 4) / (m_i * 9) (equal weights)
    ratio = Fr(float(a["kinetic_J"][0])) / Fr(float(a["kinetic_J"][1]))
    want = (Fr(W.M_E) * 4) / (Fr(W.M_DP) * 9)
    assert abs(ratio / want - 1) < Fr(1, 2**50)


@pytest.mark.parametrize("bc", [0, 1])
def test_field_energy_is_half_eps0_area_dx_sum_g_E2(bc):
    nc, dx, area = 8, 0.25, 0.5
    w = _two_species(nc, dx, bc, [0.3], [(0.0, 0.0, 0.0)], [0], area=area)
    o = O.Oracle(w)
    cases = []
    cases.append(np.full(nc + 1, 3.0))                       # uniform field
    e = np.zeros(nc + 1); e[0] = 5.0; cases.append(e)        # a single wall node
    e = np.zeros(nc + 1); e[3] = -2.0; cases.append(e)       # a single interior node
    e = np.arange(nc + 1, dtype=np.float64) - 2.5; cases.append(e)
    for E in cases:
        if not bc:
            E = E.copy(); E[nc] = E[0]                       # periodic: index nc is the ghost of node 0
        o.set_E(E)
        got = Fr(float(o.moments()["field_J"]))
        nodes = range(nc + 1) if bc else range(nc)           # periodic: nc nodes, all whole cells
        g = lambda j: Fr(1, 2) if (bc and j in (0, nc)) else Fr(1)
        want = Fr(1, 2) * Fr(EPS0) * Fr(area) * Fr(dx) * sum(g(j) * Fr(float(E[j])) ** 2 for j in nodes)
        assert abs(got - want) <= 8 * Fr(2) ** -52 * want, (bc, E.tolist())
    # uniform bounded field: energy = (1/2) eps0 E^2 x (volume area * nc * dx): wall half cells make it exact
    if bc:
        o.set_E(np.full(nc + 1, 3.0))
        vol = Fr(area) * nc * Fr(dx)
        assert abs(Fr(float(o.moments()["field_J"])) - Fr(1, 2) * Fr(EPS0) * 9 * vol) <= Fr(2) ** -48 * vol


def test_density_of_one_particle_on_a_node_shows_the_half_cell_factor():
    nc, dx, area, wgt = 8, 0.5, 0.25, 6.0e9
    sp = [W.Species("e", -E_CH, W.M_E, wgt)]
    vol = area * dx
    for xnode, j in ((0.0, 0), (2.0, 4)):
        w = W.make_custom(nc, dx, 1, 1e-12, sp, area=area, capacity=4, x=[xnode], vx=[0], vy=[0], vz=[0], sp=[0])
        n = O.Oracle(w).density(0)
        want = wgt / vol * (2.0 if j == 0 else 1.0)          # the wall node owns half a cell
        assert abs(n[j] - want) <= 1e-15 * want and np.count_nonzero(n) == 1, (xnode, n)
    # the right wall node can only be approached: x just below L puts all but 2^-32-ish of the charge on node nc
    w = W.make_custom(nc, dx, 1, 1e-12, sp, area=area, capacity=4, x=[np.nextafter(nc * dx, 0.0)], vx=[0], vy=[0],
                      vz=[0], sp=[0])
    n = O.Oracle(w).density(0)
    assert abs(n[nc] - 2.0 * wgt / vol) <= 1e-8 * wgt / vol
    # periodic: no half cells
    w = W.make_custom(nc, dx, 0, 1e-12, sp, area=area, capacity=4, x=[0.0], vx=[0], vy=[0], vz=[0], sp=[0])
    n = O.Oracle(w).density(0)
    assert n.shape[0] == nc and abs(n[0] - wgt / vol) <= 1e-15 * wgt / vol


@pytest.mark.parametrize("bc", [0, 1])
def test_density_integrates_to_the_number_of_real_particles(bc):
    """sum_j n_j x (cell volume, half cells at the walls) == N x weight, to the 1/Q quantisation of the deposit."""
    nc, dx, area, wgt = 32, 0.125, 2.0, 5.0e9
    sp = [W.Species("e", -E_CH, W.M_E, wgt), W.Species("D+", E_CH, W.M_DP, 2.0 * wgt)]
    rng = np.random.default_rng(11)
    N = 4000
    x = rng.random(N) * nc * dx
    tag = (rng.random(N) < 0.25).astype(np.uint8)
    w = W.make_custom(nc, dx, bc, 1e-12, sp, area=area, capacity=N + 8, x=x, vx=np.zeros(N), vy=np.zeros(N),
                      vz=np.zeros(N), sp=tag)
    o = O.Oracle(w)
    Q = o.Q()
    for s in range(2):
        n = o.density(s)
        vol = np.full(n.shape[0], area * dx)
        if bc:
            vol[0] *= 0.5; vol[-1] *= 0.5
        Ns = int((tag == s).sum())
        total = float((n * vol).sum())
        # Q = llrint(e w 2^40) quantises the weight to 1/Q relative
        assert abs(total - Ns * sp[s].weight) <= (1.0 / int(Q[s]) + 1e-12) * Ns * sp[s].weight


def test_uniform_load_gives_the_reference_density_in_the_interior():
    """Config 2's recipe: weight = n_ref area L / N_s, so the interior density is n_ref to sampling noise, and exactly
    n_ref on average (wall nodes included once the half-cell factor is applied)."""
    w = W.make_config(2, scale=1 / 64)
    o = O.Oracle(w)
    n_ref = 1e18
    for s in range(2):
        n = o.density(s)
        ppc = (w.sp == s).sum() / w.nc
        assert abs(n[1:-1].mean() / n_ref - 1.0) < 4.0 / np.sqrt(ppc * (w.nc - 1))
        vol = np.full(w.nc + 1, 1.0); vol[0] = vol[-1] = 0.5
        assert abs((n * vol).sum() / (w.nc * n_ref) - 1.0) < 1e-4   # 1/Q quantisation only
        # without the x2 the wall nodes would sit near n_ref/2: 200 particles per cell put them within 35 % of n_ref
        assert abs(n[0] / n_ref - 1.0) < 0.35 and abs(n[-1] / n_ref - 1.0) < 0.35
