"""Seeded synthetic workloads: the five configurations of BASELINE.json (`configs[0..4]`).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's
tests/bench.  It holds none of the method's arithmetic: it produces *inputs* --
grid and species parameters, caller-supplied tables (cross-sections, inverse
normal CDF), null-collision frequencies, and the initial particle arrays -- with
NumPy's own Philox bit generator.  Both sides receive the same arrays.

The paper's workloads are two closed-source BIT1 "high-density sheath" decks
(Table 3: bounded 1D domain between two absorbing walls, e + D+
(+ D), uniform vs non-uniform load); neither the decks nor particle data are
public, so these recipes stand in
for them with the same shape.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

# CODATA 2018
E_CHARGE = 1.602176634e-19
EPS0 = 8.8541878128e-12
M_E = 9.1093837015e-31
M_DP = 3.3435837724e-27
M_D = M_DP + M_E

# species process flags (mirrors include/bit1.h; values are part of the C ABI)
ELASTIC, IONISE, CX, ION_PRODUCT, ELECTRON_PRODUCT, TARGET_MAXWELLIAN = 1, 2, 4, 8, 16, 32
SRC_NONE, SRC_SELF, SRC_PAIR = 0, 1, 2

N_NORM = 65536
N_SIG = 2001
DE_EV = 0.5
E_ION = 13.6
LOTZ_A = 4.0e-18  # m^2 eV^2 (reading A15)


@dataclass
class Species:
    name: str
    q: float
    m: float
    weight: float
    flags: int = 0
    src_mode: int = SRC_NONE
    src_partner: int = -1
    src_vth: float = 0.0
    pnull: float = 0.0
    numax: float = 0.0
    recycle_to: int = -1      # NEXT-2: species born at the wall when this one is absorbed (-1 = none)
    recycle_vth: float = 0.0  # sqrt(e T_wall / m_recycle_to), m/s


@dataclass
class Workload:
    name: str
    nc: int
    dx: float
    bc: int  # 0 periodic, 1 absorbing walls
    area: float
    B: tuple
    dt: float
    species: List[Species]
    seed: int
    capacity: int
    src_lo: float
    src_hi: float
    n0: float
    vth_n: float
    E_ion: float
    m_n: float
    sig_el: np.ndarray
    sig_ion: np.ndarray
    sig_cx: np.ndarray
    dE_eV: float
    inv_norm: np.ndarray
    steps: int
    target_species: int = -1   # NEXT-2: species whose particle density is the collision target (-1: uniform n0)
    n_per: int = 0             # particles per loaded species of the recipe (also set when the arrays are skipped)
    x: np.ndarray = field(repr=False, default=None)
    vx: np.ndarray = field(repr=False, default=None)
    vy: np.ndarray = field(repr=False, default=None)
    vz: np.ndarray = field(repr=False, default=None)
    sp: np.ndarray = field(repr=False, default=None)
    note: str = ""

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    @property
    def L(self) -> float:
        return self.nc * self.dx

    @property
    def ng(self) -> int:
        return self.nc + 1 if self.bc else self.nc


def inv_norm_table(n_norm: int = N_NORM) -> np.ndarray:
    """Phi^-1 at clamp(i/n, 2^-17, 1-2^-17), i = 0..n (reading A18)."""
    from scipy.special import ndtri

    p = np.arange(n_norm + 1, dtype=np.float64) / n_norm
    p = np.clip(p, 2.0**-17, 1.0 - 2.0**-17)
    return np.ascontiguousarray(ndtri(p))


def sigma_tables(n_sig: int = N_SIG, dE: float = DE_EV):
    """Constant elastic 1e-19 m^2, Lotz-form ionisation (threshold 13.6 eV),
    constant charge exchange 5e-19 m^2 (BASELINE.json configs[2], reading A15)."""
    E = np.arange(n_sig, dtype=np.float64) * dE
    sig_el = np.full(n_sig, 1.0e-19)
    sig_ion = np.zeros(n_sig)
    above = E > E_ION
    sig_ion[above] = LOTZ_A * np.log(E[above] / E_ION) / (E[above] * E_ION)
    sig_cx = np.full(n_sig, 5.0e-19)
    return sig_el, sig_ion, sig_cx


def _plasma_scales(n_ref: float, Te_eV: float):
    lam = math.sqrt(EPS0 * Te_eV / (n_ref * E_CHARGE))
    wpe = math.sqrt(n_ref * E_CHARGE**2 / (EPS0 * M_E))
    return lam, wpe


def _vth(T_eV: float, m: float) -> float:
    return math.sqrt(E_CHARGE * T_eV / m)


def _null_rates(flags: int, m: float, n0: float, dt: float, tabs, dE: float):
    """numax = max over the table nodes of n0 * sum_k sigma_k(E) * g(E);
    pnull = 1 - exp(-numax dt) (reading A17)."""
    sig_el, sig_ion, sig_cx = tabs
    E = np.arange(sig_el.shape[0], dtype=np.float64) * dE
    g = np.sqrt(2.0 * E * E_CHARGE / m)
    tot = np.zeros_like(E)
    if flags & ELASTIC:
        tot += sig_el
    if flags & IONISE:
        tot += sig_ion
    if flags & CX:
        tot += sig_cx
    numax = float(np.max(n0 * tot * g))
    pnull = float(-math.expm1(-numax * dt))
    return numax, pnull


def _positions(rng, n: int, L: float, profile: str) -> np.ndarray:
    u = rng.random(n)
    if profile == "uniform":
        x = u * L
    elif profile == "exp":  # n(x) ~ exp(-|x-xc|/Ls), Ls = 0.1 L, truncated to [0, L)
        Ls = 0.1 * L
        side = rng.random(n) < 0.5
        d = -Ls * np.log1p(-u * (-math.expm1(-0.5 * L / Ls)))
        x = np.where(side, 0.5 * L + d, 0.5 * L - d)
    elif profile == "gauss":  # sigma = 0.2 L about L/2, truncated to [0, L)
        from scipy.special import ndtr, ndtri

        lo, hi = ndtr(-2.5), ndtr(2.5)
        x = 0.5 * L + 0.2 * L * ndtri(lo + u * (hi - lo))
    else:
        raise ValueError(profile)
    return np.clip(x, 0.0, np.nextafter(L, 0.0))


def profile_mean_over_peak(profile: str) -> float:
    if profile == "uniform":
        return 1.0
    if profile == "exp":
        return 0.2 * (-math.expm1(-5.0))
    if profile == "gauss":
        return 0.2 * math.sqrt(2.0 * math.pi) * math.erf(2.5 / math.sqrt(2.0))
    raise ValueError(profile)


_CFG = {
    # id: nc, N, n_ref, T_eV, bc, B(T), angle(deg), profile, nspecies, collisions, steps
    1: dict(nc=1024, N=204800, n_ref=1e18, T=10.0, bc=0, B=0.0, ang=0.0, profile="uniform", ns=2, coll=False, steps=100),
    2: dict(nc=4096, N=1638400, n_ref=1e18, T=20.0, bc=1, B=2.0, ang=2.0, profile="uniform", ns=2, coll=False, steps=1000),
    3: dict(nc=16384, N=10_000_000, n_ref=1e18, T=20.0, bc=1, B=2.0, ang=2.0, profile="uniform", ns=2, coll=True, steps=1000),
    4: dict(nc=65536, N=200_000_000, n_ref=1e18, T=20.0, bc=1, B=2.0, ang=2.0, profile="exp", ns=3, coll=True, steps=500),
    5: dict(nc=1048576, N=1_000_000_000, n_ref=1e19, T=20.0, bc=1, B=2.0, ang=3.0, profile="gauss", ns=3, coll=True, steps=100),
}


def make_config(cfg: int, scale: float = 1.0, *, n0_scale: float = 1.0, pair_source: bool = False, recycle: bool = False,
                gen_seed: Optional[int] = None, lib_seed: Optional[int] = None,
                capacity_factor: float = 1.02, particles: bool = True, ppc_scale: float = 1.0,
                quiet: bool = True) -> Workload:
    """Build configuration `cfg` (1..5) of BASELINE.json.

    scale       shrinks N and nc together (same particles per cell, same profile shape).
    n0_scale    multiplies the neutral density (tests use it to make collisions frequent).
    pair_source config 2 validation variant "2P" (reading A9): electrons SRC_NONE,
                D+ SRC_PAIR(e).
    recycle     NEXT-2: absorbed D+ ions leave a D neutral at the wall; configs without a neutral
                species get an (initially empty) one.
    particles   False skips the particle arrays (only parameters and tables).
    ppc_scale   multiplies the particles per cell at unchanged nc (the weight follows, so the physical density stays):
                e.g. configs[4]'s 1 048 576 cells with 16 instead of 954 particles per cell.
    quiet       True (default): every D+ ion is loaded on its electron (rho == 0 at step 0); False: the charged
                species are loaded independently -- the stress variant with a sqrt(N) charge imbalance, strong
                Langmuir oscillations and orders of magnitude more far movers.
    """
    c = _CFG[cfg]
    nc = max(8, int(round(c["nc"] * scale)))
    ns = c["ns"]
    n_per = max(1, int(round(c["N"] * scale * ppc_scale)) // ns)
    lam, wpe = _plasma_scales(c["n_ref"], c["T"])
    dx = 0.5 * lam
    dt = 0.1 / wpe
    L = nc * dx
    area = 1.0
    ang = math.radians(c["ang"])
    B = (c["B"] * math.cos(ang), c["B"] * math.sin(ang), 0.0) if c["B"] else (0.0, 0.0, 0.0)
    weight = c["n_ref"] * area * L * profile_mean_over_peak(c["profile"]) / n_per
    tabs = sigma_tables()
    n0 = 1e19 * n0_scale if c["coll"] else 0.0
    T0 = 1.0
    T = c["T"]
    src = SRC_SELF if c["bc"] else SRC_NONE

    fe = (ELASTIC | IONISE | ELECTRON_PRODUCT) if c["coll"] else 0
    fi = (CX | ION_PRODUCT | TARGET_MAXWELLIAN) if c["coll"] else 0
    sp = [
        Species("e", -E_CHARGE, M_E, weight, fe, src, -1, _vth(T, M_E)),
        Species("D+", +E_CHARGE, M_DP, weight, fi, src, -1, _vth(T, M_DP)),
    ]
    if ns == 3:
        sp.append(Species("D", 0.0, M_D, weight, 0, src, -1, _vth(T0, M_D)))
    if recycle and c["bc"]:
        if len(sp) == 2:
            sp.append(Species("D", 0.0, M_D, weight, 0, src, -1, _vth(T0, M_D)))
        sp[1].recycle_to = 2
        sp[1].recycle_vth = _vth(T0, M_D)
    if pair_source:
        sp[0].src_mode = SRC_NONE
        sp[1].src_mode = SRC_PAIR
        sp[1].src_partner = 0
    for s in sp:
        if s.flags & (ELASTIC | IONISE | CX):
            s.numax, s.pnull = _null_rates(s.flags, s.m, n0, dt, tabs, DE_EV)

    n_total = n_per * ns
    cap = int(math.ceil(n_total * capacity_factor)) + 1024
    w = Workload(
        name=f"c{cfg}" + ("P" if pair_source else "") + (f"@{scale:g}" if scale != 1.0 else "") +
        (f"x{ppc_scale:g}ppc" if ppc_scale != 1.0 else "") + ("" if quiet else "-noisy"),
        nc=nc, dx=dx, bc=c["bc"], area=area, B=B, dt=dt, species=sp,
        seed=(lib_seed if lib_seed is not None else 2606285340000 + cfg),
        capacity=cap, src_lo=0.25 * L, src_hi=0.75 * L, n0=n0, vth_n=_vth(T0, M_D),
        E_ion=E_ION, m_n=M_D, sig_el=tabs[0], sig_ion=tabs[1], sig_cx=tabs[2], dE_eV=DE_EV,
        inv_norm=inv_norm_table(), steps=c["steps"], n_per=n_per,
        note=f"BASELINE.json configs[{cfg - 1}], scale {scale:g}",
    )
    if not particles:
        return w
    gseed = gen_seed if gen_seed is not None else 2606285340 + cfg
    xs, vxs, vys, vzs, tags = [], [], [], [], []
    x_e = None
    for k, s in enumerate(sp[:ns]):   # a neutral species added for recycling starts empty
        Tk = T0 if s.name == "D" else T
        x, vx, vy, vz = _species_arrays(gseed, k, n_per, L, c["profile"], _vth(Tk, s.m))
        if k == 1 and quiet:
            # quiet, quasi-neutral start: every ion is loaded on its electron, rho == 0 at step 0 (SURVEY 8(d) for
            # config 1; extended to every config -- DESIGN.md "Input recipe": independent random loads leave a
            # sqrt(N) charge imbalance over 1e4..5e5 Debye lengths, i.e. Langmuir oscillations of many thermal
            # speeds that no sheath deck starts from)
            x = x_e.copy()
        if k == 0:
            x_e = x
        xs.append(x); vxs.append(vx); vys.append(vy); vzs.append(vz)
        tags.append(np.full(n_per, k, dtype=np.uint8))
    w.x = np.ascontiguousarray(np.concatenate(xs))
    w.vx = np.ascontiguousarray(np.concatenate(vxs))
    w.vy = np.ascontiguousarray(np.concatenate(vys))
    w.vz = np.ascontiguousarray(np.concatenate(vzs))
    w.sp = np.ascontiguousarray(np.concatenate(tags))
    return w


def device_particles(w: Workload, cfg: int, device, gen_seed: Optional[int] = None):
    """The particle arrays of make_config(cfg, particles=False) generated on the GPU by torch's own seeded generator
    (same profile, temperatures, equal thirds/halves per species, quiet start), as CUDA tensors (x, vx, vy, vz, sp) for
    bit1_load_particles(..., ptrs_on_device=1).  For the 1e9-particle configs[4] in bench.py: generating and pinning
    33 GB on the host would take minutes; nothing is compared with the oracle on these arrays (full-size parity runs
    use make_config's host arrays)."""
    import torch

    c = _CFG[cfg]
    ns = c["ns"]
    n_per = w.n_per
    n = n_per * ns
    g = torch.Generator(device=device)
    g.manual_seed((gen_seed if gen_seed is not None else 2606285340 + cfg) & (2**63 - 1))
    x = torch.empty(n, dtype=torch.float64, device=device)
    v = [torch.empty(n, dtype=torch.float64, device=device) for _ in range(3)]
    sp = torch.empty(n, dtype=torch.uint8, device=device)
    L = w.L
    step = 1 << 25
    for k in range(ns):
        Tk = 1.0 if w.species[k].name == "D" else c["T"]
        vth = _vth(Tk, w.species[k].m)
        lo = k * n_per
        sp[lo:lo + n_per] = k
        for a in range(0, n_per, step):
            m = min(step, n_per - a)
            sl = slice(lo + a, lo + a + m)
            if k == 1:
                x[sl] = x[a:a + m]          # quiet start: every ion on its electron
            else:
                u = torch.rand(m, dtype=torch.float64, device=device, generator=g)
                if c["profile"] == "uniform":
                    xs = u * L
                elif c["profile"] == "exp":
                    Ls = 0.1 * L
                    side = torch.rand(m, dtype=torch.float64, device=device, generator=g) < 0.5
                    d = -Ls * torch.log1p(-u * (-math.expm1(-0.5 * L / Ls)))
                    xs = torch.where(side, 0.5 * L + d, 0.5 * L - d)
                else:
                    plo = 0.5 * (1.0 + math.erf(-2.5 / math.sqrt(2.0)))
                    phi = 0.5 * (1.0 + math.erf(2.5 / math.sqrt(2.0)))
                    xs = 0.5 * L + 0.2 * L * math.sqrt(2.0) * torch.special.erfinv(2.0 * (plo + u * (phi - plo)) - 1.0)
                x[sl] = torch.clamp(xs, 0.0, float(np.nextafter(L, 0.0)))
            for comp in v:
                comp[sl] = vth * torch.randn(m, dtype=torch.float64, device=device, generator=g)
    return x, v[0], v[1], v[2], sp


_CHUNK = 1 << 21


def _species_arrays(gseed: int, k: int, n: int, L: float, profile: str, vth: float):
    """Positions and velocities of one species, generated in fixed chunks of 2^21 particles, each chunk from
    its own Philox key (gseed, species, chunk) -- the arrays do not depend on how many threads fill them."""
    from concurrent.futures import ThreadPoolExecutor
    import os

    x = np.empty(n); vx = np.empty(n); vy = np.empty(n); vz = np.empty(n)

    def fill(j):
        lo, hi = j * _CHUNK, min(n, (j + 1) * _CHUNK)
        rng = np.random.Generator(np.random.Philox(key=[gseed, (k << 32) | j]))
        x[lo:hi] = _positions(rng, hi - lo, L, profile)
        vx[lo:hi] = vth * rng.standard_normal(hi - lo)
        vy[lo:hi] = vth * rng.standard_normal(hi - lo)
        vz[lo:hi] = vth * rng.standard_normal(hi - lo)

    nchunks = (n + _CHUNK - 1) // _CHUNK
    if nchunks <= 1:
        fill(0)
    else:
        with ThreadPoolExecutor(max_workers=min(32, os.cpu_count() or 1)) as ex:
            list(ex.map(fill, range(nchunks)))
    return x, vx, vy, vz


def make_custom(nc: int, dx: float, bc: int, dt: float, species: List[Species], *, B=(0.0, 0.0, 0.0),
                area: float = 1.0, seed: int = 1, capacity: int = 1024, n0: float = 0.0,
                T0_eV: float = 1.0, src_lo: Optional[float] = None, src_hi: Optional[float] = None,
                x=None, vx=None, vy=None, vz=None, sp=None, name: str = "custom", tabs=None) -> Workload:
    """Small hand-made workloads for unit tests (single particles, beams, cold plasma)."""
    tabs = tabs if tabs is not None else sigma_tables()
    L = nc * dx
    for s in species:
        if s.flags & (ELASTIC | IONISE | CX) and s.numax == 0.0:
            s.numax, s.pnull = _null_rates(s.flags, s.m, n0, dt, tabs, DE_EV)
    w = Workload(
        name=name, nc=nc, dx=dx, bc=bc, area=area, B=tuple(B), dt=dt, species=species, seed=seed,
        capacity=capacity, src_lo=(0.25 * L if src_lo is None else src_lo),
        src_hi=(0.75 * L if src_hi is None else src_hi), n0=n0, vth_n=_vth(T0_eV, M_D), E_ion=E_ION,
        m_n=M_D, sig_el=tabs[0], sig_ion=tabs[1], sig_cx=tabs[2], dE_eV=DE_EV,
        inv_norm=inv_norm_table(), steps=1,
    )
    f8 = lambda a: np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if x is not None:
        w.x, w.vx, w.vy, w.vz = f8(x), f8(vx), f8(vy), f8(vz)
        w.sp = np.ascontiguousarray(np.asarray(sp, dtype=np.uint8))
    return w
