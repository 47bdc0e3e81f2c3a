"""ctypes wrapper around oracle/bit1_oracle.c -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It imports nothing from paper_2606_28534_b200: a workload
is taken duck-typed (any object with the attributes of workloads.Workload).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bit1_oracle.c")
_LIB = os.path.join(_HERE, "libbit1_oracle.so")
_lib = None

c_f64p = C.POINTER(C.c_double)
c_i64p = C.POINTER(C.c_int64)
c_u64p = C.POINTER(C.c_uint64)
c_i32p = C.POINTER(C.c_int32)
c_u32p = C.POINTER(C.c_uint32)
c_u8p = C.POINTER(C.c_uint8)


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off: one IEEE operation per written operation."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int32, C.c_double, C.c_int32, C.c_double, c_f64p, C.c_double,
                                 C.c_int32, c_f64p, c_f64p, c_f64p, c_u32p, c_i32p, c_i32p, c_f64p,
                                 c_f64p, c_f64p, C.c_uint64, C.c_uint64, C.c_double, C.c_double,
                                 C.c_double, C.c_double, C.c_double, C.c_double, c_f64p, c_f64p,
                                 c_f64p, C.c_int32, C.c_double, c_f64p, C.c_int32]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_load.restype = C.c_int
        L.orc_load.argtypes = [C.c_void_p, C.c_uint64, c_f64p, c_f64p, c_f64p, c_f64p, c_u8p, c_u32p]
        L.orc_restore.restype = C.c_int
        L.orc_restore.argtypes = [C.c_void_p, C.c_uint64, c_f64p, c_f64p, c_f64p, c_f64p, c_i32p,
                                  c_u32p, c_u8p, C.c_uint64, C.c_uint32, c_u64p, c_i64p]
        L.orc_step.argtypes = [C.c_void_p, C.c_uint64, C.c_int]
        for name in ("orc_phase_push", "orc_phase_sort", "orc_phase_deposit", "orc_phase_field"):
            getattr(L, name).argtypes = [C.c_void_p]
        L.orc_n.restype = C.c_uint64
        L.orc_n.argtypes = [C.c_void_p]
        L.orc_n_slots.restype = C.c_uint64
        L.orc_n_slots.argtypes = [C.c_void_p]
        L.orc_step_index.restype = C.c_uint64
        L.orc_step_index.argtypes = [C.c_void_p]
        L.orc_next_pid.restype = C.c_uint32
        L.orc_next_pid.argtypes = [C.c_void_p]
        L.orc_flagword.restype = C.c_uint32
        L.orc_flagword.argtypes = [C.c_void_p]
        L.orc_set_step.argtypes = [C.c_void_p, C.c_uint64]
        L.orc_set_E.argtypes = [C.c_void_p, c_f64p]
        L.orc_get_particles.argtypes = [C.c_void_p, c_f64p, c_f64p, c_f64p, c_f64p, c_i32p, c_u32p, c_u8p]
        L.orc_get_cell_start.argtypes = [C.c_void_p, c_i64p]
        L.orc_get_rho.argtypes = [C.c_void_p, c_i64p]
        L.orc_get_dens.argtypes = [C.c_void_p, c_i64p]
        L.orc_get_phi.argtypes = [C.c_void_p, c_f64p]
        L.orc_get_E.argtypes = [C.c_void_p, c_f64p]
        L.orc_get_Q.argtypes = [C.c_void_p, c_i64p]
        L.orc_get_wall.argtypes = [C.c_void_p, c_u64p, c_i64p]
        L.orc_get_diag.argtypes = [C.c_void_p, c_u64p, c_u64p, c_u64p]
        L.orc_get_constants.argtypes = [C.c_void_p, c_f64p, c_f64p, c_f64p, c_f64p]
        L.orc_get_density.argtypes = [C.c_void_p, C.c_int, c_f64p]
        L.orc_get_moments.argtypes = [C.c_void_p, c_u64p, c_f64p, c_f64p, c_f64p]
        L.orc_poisson.argtypes = [C.c_int32, C.c_int32, C.c_double, C.c_double, c_i64p, c_f64p, c_f64p]
        L.orc_smooth121.argtypes = [C.c_int32, C.c_int32, c_i64p, c_i64p]
        L.orc_set_smoothing.argtypes = [C.c_void_p, C.c_int32]
        L.orc_set_recycling.restype = C.c_int
        L.orc_set_recycling.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double]
        L.orc_set_neutral_target.restype = C.c_int
        L.orc_set_neutral_target.argtypes = [C.c_void_p, C.c_int32]
        L.orc_recycled.restype = C.c_uint64
        L.orc_recycled.argtypes = [C.c_void_p]
        L.orc_set_averaging.restype = C.c_int
        L.orc_set_averaging.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        L.orc_get_average.argtypes = [C.c_void_p, c_i64p, c_f64p, c_u64p, c_u64p]
        L.orc_get_rho_smoothed.argtypes = [C.c_void_p, c_i64p]
        L.orc_philox4x32_10.argtypes = [c_u32p, c_u32p, c_u32p]
        L.orc_u53.restype = C.c_double
        L.orc_u53.argtypes = [C.c_uint32, C.c_uint32]
        L.orc_u32.restype = C.c_double
        L.orc_u32.argtypes = [C.c_uint32]
        L.orc_normal.restype = C.c_double
        L.orc_normal.argtypes = [C.c_void_p, C.c_uint32]
        L.orc_direction.restype = C.c_int
        L.orc_direction.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_uint32, c_f64p]
        L.orc_sigma.restype = C.c_double
        L.orc_sigma.argtypes = [C.c_void_p, C.c_int, C.c_double]
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def _f8(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, c_u32p), _p(k, c_u32p), _p(out, c_u32p))
    return out


def u53(a, b):
    return lib().orc_u53(int(a), int(b))


def u32(a):
    return lib().orc_u32(int(a))


def poisson(nc, bc, Kphi, KE, rho):
    rho = np.ascontiguousarray(np.asarray(rho, dtype=np.int64))
    phi = np.zeros(nc + 1)
    E = np.zeros(nc + 1)
    lib().orc_poisson(nc, bc, Kphi, KE, _p(rho, c_i64p), _p(phi, c_f64p), _p(E, c_f64p))
    return phi, E


def smooth121(nc, bc, rho):
    """One 1-2-1 pass in exact integers: returns 4 x the smoothed array (reading N1-a)."""
    rho = np.ascontiguousarray(np.asarray(rho, dtype=np.int64))
    out = np.zeros_like(rho)
    lib().orc_smooth121(nc, bc, _p(rho, c_i64p), _p(out, c_i64p))
    return out


class Oracle:
    """One oracle simulation built from a workload description."""

    def __init__(self, w, load: bool = True):
        L = lib()
        self.w = w
        self.ns = len(w.species)
        self.nc, self.bc = int(w.nc), int(w.bc)
        self.ng = self.nc + 1 if self.bc else self.nc
        sp = w.species
        arr = lambda f, dt=np.float64: np.ascontiguousarray(np.array([getattr(s, f) for s in sp], dtype=dt))
        q, m, wt = arr("q"), arr("m"), arr("weight")
        fl, sm, spn = arr("flags", np.uint32), arr("src_mode", np.int32), arr("src_partner", np.int32)
        sv, pn, nm = arr("src_vth"), arr("pnull"), arr("numax")
        B = _f8(w.B)
        sig_el, sig_ion, sig_cx, inv_norm = _f8(w.sig_el), _f8(w.sig_ion), _f8(w.sig_cx), _f8(w.inv_norm)
        self.h = L.orc_create(self.nc, w.dx, self.bc, w.area, _p(B, c_f64p), w.dt, self.ns,
                              _p(q, c_f64p), _p(m, c_f64p), _p(wt, c_f64p), _p(fl, c_u32p),
                              _p(sm, c_i32p), _p(spn, c_i32p), _p(sv, c_f64p), _p(pn, c_f64p),
                              _p(nm, c_f64p), int(w.seed), int(w.capacity), w.src_lo, w.src_hi, w.n0,
                              w.vth_n, w.E_ion, w.m_n, _p(sig_el, c_f64p), _p(sig_ion, c_f64p),
                              _p(sig_cx, c_f64p), int(sig_el.shape[0]), w.dE_eV, _p(inv_norm, c_f64p),
                              int(inv_norm.shape[0] - 1))
        if not self.h:
            raise ValueError("orc_create rejected the configuration")
        if getattr(w, "target_species", -1) >= 0:
            self.set_neutral_target(w.target_species)
        for k, spc in enumerate(sp):
            if getattr(spc, "recycle_to", -1) >= 0:
                self.set_recycling(k, spc.recycle_to, spc.recycle_vth)
        if load and w.x is not None:
            self.load(w.x, w.vx, w.vy, w.vz, w.sp)

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_destroy(self.h)
            self.h = None

    # -- state in -----------------------------------------------------
    def load(self, x, vx, vy, vz, sp, pid=None):
        x, vx, vy, vz = _f8(x), _f8(vx), _f8(vy), _f8(vz)
        sp = np.ascontiguousarray(np.asarray(sp, dtype=np.uint8))
        pp = None
        if pid is not None:
            pid = np.ascontiguousarray(np.asarray(pid, dtype=np.uint32))
            pp = _p(pid, c_u32p)
        rc = lib().orc_load(self.h, x.shape[0], _p(x, c_f64p), _p(vx, c_f64p), _p(vy, c_f64p),
                            _p(vz, c_f64p), _p(sp, c_u8p), pp)
        if rc:
            raise ValueError(f"orc_load failed rc={rc}")

    def restore(self, st):
        """st: dict from snapshot()."""
        wc = np.ascontiguousarray(st["wall_count"].astype(np.uint64))
        wq = np.ascontiguousarray(st["wall_charge"].astype(np.int64))
        rc = lib().orc_restore(self.h, st["x"].shape[0], _p(st["x"], c_f64p), _p(st["vx"], c_f64p),
                               _p(st["vy"], c_f64p), _p(st["vz"], c_f64p), _p(st["cell"], c_i32p),
                               _p(st["pid"], c_u32p), _p(st["sp"], c_u8p), int(st["step"]),
                               int(st["next_pid"]), _p(wc, c_u64p), _p(wq, c_i64p))
        if rc:
            raise ValueError(f"orc_restore failed rc={rc}")

    def snapshot(self):
        st = self.particles()
        wc, wq = self.wall()
        st.update(step=self.step_index, next_pid=self.next_pid, wall_count=wc, wall_charge=wq)
        return st

    # -- stepping -----------------------------------------------------
    def step(self, n=1, freeze_field=False):
        lib().orc_step(self.h, int(n), int(bool(freeze_field)))

    def phase_push(self):
        lib().orc_phase_push(self.h)

    def phase_sort(self):
        lib().orc_phase_sort(self.h)

    def phase_deposit(self):
        lib().orc_phase_deposit(self.h)

    def phase_field(self):
        lib().orc_phase_field(self.h)

    def set_E(self, E):
        E = _f8(E)
        assert E.shape[0] == self.nc + 1
        lib().orc_set_E(self.h, _p(E, c_f64p))

    def set_step(self, s):
        lib().orc_set_step(self.h, int(s))

    # -- state out ----------------------------------------------------
    @property
    def n(self):
        return int(lib().orc_n(self.h))

    @property
    def n_slots(self):
        return int(lib().orc_n_slots(self.h))

    @property
    def step_index(self):
        return int(lib().orc_step_index(self.h))

    @property
    def next_pid(self):
        return int(lib().orc_next_pid(self.h))

    @property
    def flagword(self):
        return int(lib().orc_flagword(self.h))

    def particles(self):
        n = self.n_slots
        d = dict(x=np.zeros(n), vx=np.zeros(n), vy=np.zeros(n), vz=np.zeros(n),
                 cell=np.zeros(n, np.int32), pid=np.zeros(n, np.uint32), sp=np.zeros(n, np.uint8))
        lib().orc_get_particles(self.h, _p(d["x"], c_f64p), _p(d["vx"], c_f64p), _p(d["vy"], c_f64p),
                                _p(d["vz"], c_f64p), _p(d["cell"], c_i32p), _p(d["pid"], c_u32p),
                                _p(d["sp"], c_u8p))
        return d

    def particle_array(self, name):
        """One of x, vx, vy, vz, cell, pid, sp alone (the others are not copied): for states too large to hold twice."""
        order = ["x", "vx", "vy", "vz", "cell", "pid", "sp"]
        dt = dict(x=np.float64, vx=np.float64, vy=np.float64, vz=np.float64, cell=np.int32, pid=np.uint32, sp=np.uint8)
        ct = dict(x=c_f64p, vx=c_f64p, vy=c_f64p, vz=c_f64p, cell=c_i32p, pid=c_u32p, sp=c_u8p)
        a = np.zeros(self.n_slots, dt[name])
        args = [None] * 7
        args[order.index(name)] = _p(a, ct[name])
        lib().orc_get_particles(self.h, *args)
        return a

    def cell_start(self):
        cs = np.zeros(self.nc + 1, np.int64)
        lib().orc_get_cell_start(self.h, _p(cs, c_i64p))
        return cs

    def rho(self):
        r = np.zeros(self.ng, np.int64)
        lib().orc_get_rho(self.h, _p(r, c_i64p))
        return r

    def set_neutral_target(self, species: int):
        assert lib().orc_set_neutral_target(self.h, int(species)) == 0

    def set_recycling(self, s: int, to: int, vth: float):
        assert lib().orc_set_recycling(self.h, int(s), int(to), float(vth)) == 0

    @property
    def recycled(self):
        return int(lib().orc_recycled(self.h))

    def set_smoothing(self, passes: int):
        lib().orc_set_smoothing(self.h, int(passes))

    def set_averaging(self, window: int, interval: int):
        assert lib().orc_set_averaging(self.h, int(window), int(interval)) == 0

    def average(self):
        """Latest latched window: (dens_sum[ns, ng] int64, phi_sum[nc+1], count, step)."""
        d = np.zeros((self.ns, self.ng), np.int64)
        f = np.zeros(self.nc + 1)
        cnt = np.zeros(1, np.uint64)
        st = np.zeros(1, np.uint64)
        lib().orc_get_average(self.h, _p(d, c_i64p), _p(f, c_f64p), _p(cnt, c_u64p), _p(st, c_u64p))
        return d, f, int(cnt[0]), int(st[0])

    def rho_smoothed(self):
        r = np.zeros(self.ng, np.int64)
        lib().orc_get_rho_smoothed(self.h, _p(r, c_i64p))
        return r

    def dens(self):
        d = np.zeros((self.ns, self.ng), np.int64)
        lib().orc_get_dens(self.h, _p(d, c_i64p))
        return d

    def phi(self):
        a = np.zeros(self.nc + 1)
        lib().orc_get_phi(self.h, _p(a, c_f64p))
        return a

    def E(self):
        a = np.zeros(self.nc + 1)
        lib().orc_get_E(self.h, _p(a, c_f64p))
        return a

    def Q(self):
        a = np.zeros(self.ns, np.int64)
        lib().orc_get_Q(self.h, _p(a, c_i64p))
        return a

    def wall(self):
        cnt = np.zeros((2, self.ns), np.uint64)
        chg = np.zeros(2, np.int64)
        lib().orc_get_wall(self.h, _p(cnt, c_u64p), _p(chg, c_i64p))
        return cnt, chg

    def diag(self):
        d5 = np.zeros(5, np.uint64)
        cand = np.zeros(self.ns, np.uint64)
        ev = np.zeros((self.ns, 3), np.uint64)
        lib().orc_get_diag(self.h, _p(d5, c_u64p), _p(cand, c_u64p), _p(ev, c_u64p))
        return dict(nu_overflow=int(d5[0]), dir_fallback=int(d5[1]), escape=int(d5[2]),
                    births=int(d5[3]), reinject=int(d5[4]), candidates=cand, events=ev)

    def constants(self):
        out = np.zeros(4)
        h = np.zeros(self.ns)
        t3 = np.zeros((self.ns, 3))
        s3 = np.zeros((self.ns, 3))
        lib().orc_get_constants(self.h, _p(out, c_f64p), _p(h, c_f64p), _p(t3, c_f64p), _p(s3, c_f64p))
        return dict(inv_dx=out[0], L=out[1], Kphi=out[2], KE=out[3], h=h, t=t3, s=s3)

    def density(self, s):
        a = np.zeros(self.ng)
        lib().orc_get_density(self.h, int(s), _p(a, c_f64p))
        return a

    def moments(self):
        cnt = np.zeros(self.ns, np.uint64)
        ke = np.zeros(self.ns)
        px = np.zeros(self.ns)
        fe = np.zeros(1)
        lib().orc_get_moments(self.h, _p(cnt, c_u64p), _p(ke, c_f64p), _p(px, c_f64p), _p(fe, c_f64p))
        return dict(count=cnt, kinetic_J=ke, px=px, field_J=float(fe[0]))

    def normal(self, word):
        return lib().orc_normal(self.h, int(word))

    def direction(self, pid, step, first_slot):
        n = np.zeros(3)
        fb = lib().orc_direction(self.h, int(pid), int(step), int(first_slot), _p(n, c_f64p))
        return n, fb

    def sigma(self, which, E_eV):
        return lib().orc_sigma(self.h, int(which), float(E_eV))
