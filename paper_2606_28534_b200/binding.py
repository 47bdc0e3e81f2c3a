"""Thin Python binding of libbit1 (include/bit1.h): argument marshalling only.

Same names as the C ABI.  PyTorch supplies device memory (the workspace tensor) and CUDA streams; every
step of the hot path runs in the library's kernels.  There is no CPU fallback: if libbit1.so is missing
or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

MAX_SPECIES = 8
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbit1.so")

OK, ERR_INVALID_ARG, ERR_RANGE, ERR_CAPACITY, ERR_STATE, ERR_CUDA, ERR_CHECKPOINT, ERR_DEVICE_FLAG = range(8)
ERR_STATIC_LIMIT = 8
FIELD_STATIC_MAX_CELLS = 1 << 20   # BIT1_FIELD_STATIC_MAX_CELLS
FLAG_CAPACITY, FLAG_ESCAPE, FLAG_PID_WRAP = 1, 2, 8

c_f64p = C.POINTER(C.c_double)


class bit1_grid(C.Structure):
    _fields_ = [("nc", C.c_int32), ("bc", C.c_int32), ("dx", C.c_double), ("area", C.c_double),
                ("Bx", C.c_double), ("By", C.c_double), ("Bz", C.c_double)]


class bit1_species(C.Structure):
    _fields_ = [("q", C.c_double), ("m", C.c_double), ("weight", C.c_double), ("flags", C.c_uint32),
                ("src_mode", C.c_int32), ("src_partner", C.c_int32), ("_pad", C.c_int32),
                ("src_vth", C.c_double), ("pnull", C.c_double), ("numax", C.c_double)]


class bit1_options(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("capacity", C.c_uint64), ("src_lo", C.c_double), ("src_hi", C.c_double),
                ("n0", C.c_double), ("vth_n", C.c_double), ("E_ion", C.c_double), ("m_n", C.c_double),
                ("sig_el", c_f64p), ("sig_ion", c_f64p), ("sig_cx", c_f64p), ("n_sig", C.c_int32),
                ("n_norm", C.c_int32), ("dE_eV", C.c_double), ("inv_norm", c_f64p), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t), ("compute_stream", C.c_void_p), ("side_stream", C.c_void_p),
                ("checkpoint_staging", C.c_int32), ("launch_mode", C.c_int32), ("window_radius_max", C.c_int32),
                ("window_radius_fixed", C.c_int32), ("side_list_capacity", C.c_uint64)]


class bit1_moments(C.Structure):
    _fields_ = [("step", C.c_uint64), ("n_live", C.c_uint64), ("count", C.c_uint64 * MAX_SPECIES),
                ("kinetic_J", C.c_double * MAX_SPECIES), ("px", C.c_double * MAX_SPECIES), ("field_J", C.c_double),
                ("wall_count", (C.c_uint64 * MAX_SPECIES) * 2), ("wall_charge_fixed", C.c_int64 * 2),
                ("rho_total_fixed", C.c_int64), ("flags", C.c_uint32), ("next_pid", C.c_uint32),
                ("nu_overflow", C.c_uint64), ("dir_fallback", C.c_uint64), ("escape", C.c_uint64),
                ("births", C.c_uint64), ("reinject", C.c_uint64), ("candidates", C.c_uint64 * MAX_SPECIES),
                ("events", (C.c_uint64 * 3) * MAX_SPECIES), ("far_movers", C.c_uint64),
                ("max_far_movers_per_step", C.c_uint64), ("recycled", C.c_uint64), ("general_steps", C.c_uint64),
                ("window_radius", C.c_uint32), ("check_failures", C.c_uint32), ("check_line", C.c_uint32),
                ("_pad", C.c_uint32), ("check_index", C.c_int64), ("check_limit", C.c_int64),
                ("density", c_f64p * MAX_SPECIES)]


class bit1_stream_header(C.Structure):
    _fields_ = [("magic", C.c_char * 8), ("seq_begin", C.c_uint64), ("seq", C.c_uint64), ("step", C.c_uint64),
                ("n_total", C.c_uint64), ("bytes", C.c_uint64), ("nc", C.c_int32), ("ns", C.c_int32), ("bc", C.c_int32),
                ("_pad", C.c_int32), ("count", C.c_uint64 * MAX_SPECIES), ("off_counts", C.c_uint64 * MAX_SPECIES),
                ("off_x", C.c_uint64 * MAX_SPECIES), ("off_vx", C.c_uint64 * MAX_SPECIES),
                ("off_vy", C.c_uint64 * MAX_SPECIES), ("off_vz", C.c_uint64 * MAX_SPECIES),
                ("off_pid", C.c_uint64 * MAX_SPECIES)]


_lib = None


def load_library(path: Optional[str] = None):
    """dlopen libbit1.so and declare every entry point of include/bit1.h.  Raises if it is missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or os.environ.get("BIT1_LIB") or LIB_PATH   # BIT1_LIB: a libbit1.so built with other tile geometry
    if not os.path.exists(p):
        raise RuntimeError(f"{p} not found: build it with `python -m paper_2606_28534_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(p)
    vp = C.c_void_p
    L.bit1_workspace_size.restype = C.c_size_t
    L.bit1_workspace_size.argtypes = [C.POINTER(bit1_grid), C.c_int, C.POINTER(bit1_options)]
    L.bit1_create.restype = C.c_int
    L.bit1_create.argtypes = [C.POINTER(bit1_grid), C.POINTER(bit1_species), C.c_int, C.c_double,
                              C.POINTER(bit1_options), C.POINTER(vp)]
    L.bit1_load_particles.restype = C.c_int
    L.bit1_load_particles.argtypes = [vp, C.c_uint64, vp, vp, vp, vp, vp, vp, C.c_int]
    L.bit1_step.restype = C.c_int
    L.bit1_step.argtypes = [vp, C.c_uint64]
    L.bit1_sync.restype = C.c_int
    L.bit1_sync.argtypes = [vp]
    L.bit1_get_count.restype = C.c_int
    L.bit1_get_count.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.bit1_get_rho.restype = C.c_int
    L.bit1_get_rho.argtypes = [vp, vp, vp]
    for name in ("bit1_get_phi", "bit1_get_E", "bit1_get_dens"):
        getattr(L, name).restype = C.c_int
        getattr(L, name).argtypes = [vp, vp]
    L.bit1_get_moments.restype = C.c_int
    L.bit1_get_moments.argtypes = [vp, C.POINTER(bit1_moments)]
    L.bit1_get_particles.restype = C.c_int
    L.bit1_get_particles.argtypes = [vp] + [vp] * 8
    L.bit1_set_recycling.restype = C.c_int
    L.bit1_set_recycling.argtypes = [vp, C.c_int, C.c_int, C.c_double]
    L.bit1_set_neutral_target.restype = C.c_int
    L.bit1_set_neutral_target.argtypes = [vp, C.c_int]
    L.bit1_set_smoothing.restype = C.c_int
    L.bit1_set_smoothing.argtypes = [vp, C.c_int]
    L.bit1_get_rho_smoothed.restype = C.c_int
    L.bit1_get_rho_smoothed.argtypes = [vp, vp]
    L.bit1_set_averaging.restype = C.c_int
    L.bit1_set_averaging.argtypes = [vp, C.c_int, C.c_int]
    L.bit1_get_average.restype = C.c_int
    L.bit1_get_average.argtypes = [vp, vp, vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.bit1_set_E.restype = C.c_int
    L.bit1_set_E.argtypes = [vp, vp, C.c_int]
    L.bit1_set_step.restype = C.c_int
    L.bit1_set_step.argtypes = [vp, C.c_uint64]
    L.bit1_checkpoint_size.restype = C.c_size_t
    L.bit1_checkpoint_size.argtypes = [vp]
    L.bit1_checkpoint.restype = C.c_int
    L.bit1_checkpoint.argtypes = [vp, vp, C.c_size_t, C.POINTER(C.c_size_t)]
    L.bit1_checkpoint_wait.restype = C.c_int
    L.bit1_checkpoint_wait.argtypes = [vp]
    L.bit1_restart.restype = C.c_int
    L.bit1_restart.argtypes = [vp, vp, C.c_size_t]
    L.bit1_export_species.restype = C.c_int
    L.bit1_export_species.argtypes = [vp, C.c_int, C.c_uint64, C.POINTER(C.c_uint64), vp, vp, vp, vp, vp, vp]
    L.bit1_stream_slot_size.restype = C.c_size_t
    L.bit1_stream_slot_size.argtypes = [vp]
    L.bit1_stream_open.restype = C.c_int
    L.bit1_stream_open.argtypes = [vp, vp, C.c_size_t, C.c_int]
    L.bit1_stream_publish.restype = C.c_int
    L.bit1_stream_publish.argtypes = [vp, C.POINTER(C.c_uint64)]
    L.bit1_stream_acquire.restype = C.c_int
    L.bit1_stream_acquire.argtypes = [vp, C.c_uint64, C.POINTER(vp), C.POINTER(C.c_uint64)]
    L.bit1_stream_release.restype = C.c_int
    L.bit1_stream_release.argtypes = [vp, C.c_uint64]
    L.bit1_stream_close.restype = C.c_int
    L.bit1_stream_close.argtypes = [vp]
    L.bit1_destroy.restype = None
    L.bit1_destroy.argtypes = [vp]
    L.bit1_error_string.restype = C.c_char_p
    L.bit1_error_string.argtypes = [C.c_int]
    L.bit1_profile.restype = C.c_int
    L.bit1_profile.argtypes = [vp, C.c_int]
    L.bit1_get_profile.restype = C.c_int
    L.bit1_get_profile.argtypes = [vp, C.POINTER(C.c_double * 4), C.POINTER(C.c_uint64)]
    L.bit1_launch_count.restype = C.c_uint64
    L.bit1_launch_count.argtypes = [vp]
    L.bit1_build_is_checked.restype = C.c_int
    L.bit1_build_is_checked.argtypes = []
    L.bit1_check_selftest.restype = C.c_int
    L.bit1_check_selftest.argtypes = [vp]
    L.bit1_field_solve_static.restype = C.c_int
    L.bit1_field_solve_static.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_int32, vp]
    if path is None:
        _lib = L
    return L


class Bit1Error(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = load_library().bit1_error_string(status).decode()
        super().__init__(f"{where}: {msg} (status {status})")


def _check(status: int, where: str):
    if status != OK:
        raise Bit1Error(status, where)


def _f8(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a):
    """HOST numpy array or torch tensor (host or device) -> raw pointer."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


def field_solve_static(rho, phi, E, nc: int, bc: int, dx: float, area: float, passes: int = 0, stream=None, lib=None):
    """bit1_field_solve_static: smoothing + Poisson solve of one rho array with no context and no workspace.

    For code that may not allocate GPU memory (a plug-in fed from its host's memory pool, a callback that runs while
    that pool is locked, a job with a fixed device-memory budget): the library allocates nothing in this call; its
    temporaries live in an array built into libbit1.so, which is why nc may not exceed FIELD_STATIC_MAX_CELLS
    (Bit1Error with status ERR_STATIC_LIMIT beyond it).  rho (int64[ng]), phi and E (float64[nc + 1]) are torch CUDA
    tensors the caller already owns, all on the current device; stream is a torch.cuda.Stream or None (the current
    stream).  The kernel is enqueued, not waited for.  Calls on one device share the built-in array: keep them on one
    stream (include/bit1.h has the full list of rules).  Marshalling only."""
    import torch

    L = lib if lib is not None else load_library()
    ng = nc + 1 if bc else nc
    for t, n, dt, name in ((rho, ng, torch.int64, "rho"), (phi, nc + 1, torch.float64, "phi"), (E, nc + 1, torch.float64, "E")):
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() == n):
            raise ValueError(f"{name}: need a contiguous CUDA tensor of {n} x {dt}")
    s = stream if stream is not None else torch.cuda.current_stream(rho.device)
    with torch.cuda.device(rho.device):
        st = L.bit1_field_solve_static(rho.data_ptr(), phi.data_ptr(), E.data_ptr(), int(nc), int(bc), float(dx), float(area),
                                       int(passes), s.cuda_stream)
    _check(st, "bit1_field_solve_static")


class Bit1:
    """One libbit1 context.  Methods mirror the C entry points one to one."""

    def __init__(self, w, *, checkpoint_staging: bool = False, device: str = "cuda:0", side_stream: bool = True,
                 direct_launch: bool = False, window_radius_max: int = 0, window_radius: Optional[int] = None,
                 side_list_capacity: int = 0, lib=None):
        """window_radius: None = adaptive (default), k = pinned to k cells; the other keywords are bit1_options fields.
        lib: a library from load_library(path), e.g. the checked build (default: the shipped libbit1.so)."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("libbit1 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.lib = lib if lib is not None else load_library()
        self.w = w
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.ns = len(w.species)
        self.nc, self.bc = int(w.nc), int(w.bc)
        self.ng = self.nc + 1 if self.bc else self.nc
        g = bit1_grid(self.nc, self.bc, w.dx, w.area, w.B[0], w.B[1], w.B[2])
        sp = (bit1_species * self.ns)()
        for k, s in enumerate(w.species):
            sp[k] = bit1_species(s.q, s.m, s.weight, s.flags, s.src_mode, s.src_partner, 0, s.src_vth, s.pnull,
                                 s.numax)
        o = bit1_options()
        o.seed, o.capacity = int(w.seed), int(w.capacity)
        o.checkpoint_staging = int(checkpoint_staging)
        o.launch_mode = int(direct_launch)
        o.window_radius_max = int(window_radius_max)
        o.window_radius_fixed = 0 if window_radius is None else int(window_radius) + 1
        o.side_list_capacity = int(side_list_capacity)
        nbytes = self.lib.bit1_workspace_size(C.byref(g), self.ns, C.byref(o))
        if nbytes == 0:
            raise Bit1Error(ERR_INVALID_ARG, "bit1_workspace_size")
        self.workspace_bytes = nbytes
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self.compute_stream = torch.cuda.Stream(device=self.device)
        self.side_stream = torch.cuda.Stream(device=self.device) if side_stream else None
        self._keep = [_f8(w.sig_el), _f8(w.sig_ion), _f8(w.sig_cx), _f8(w.inv_norm)]
        o.src_lo, o.src_hi = w.src_lo, w.src_hi
        o.n0, o.vth_n, o.E_ion, o.m_n = w.n0, w.vth_n, w.E_ion, w.m_n
        o.sig_el = self._keep[0].ctypes.data_as(c_f64p)
        o.sig_ion = self._keep[1].ctypes.data_as(c_f64p)
        o.sig_cx = self._keep[2].ctypes.data_as(c_f64p)
        o.n_sig = int(self._keep[0].shape[0])
        o.n_norm = int(self._keep[3].shape[0] - 1)
        o.dE_eV = w.dE_eV
        o.inv_norm = self._keep[3].ctypes.data_as(c_f64p)
        o.workspace, o.workspace_bytes = base, nbytes
        o.compute_stream = self.compute_stream.cuda_stream
        o.side_stream = self.side_stream.cuda_stream if self.side_stream is not None else None
        h = C.c_void_p()
        _check(self.lib.bit1_create(C.byref(g), sp, self.ns, w.dt, C.byref(o), C.byref(h)), "bit1_create")
        self.h = h
        if getattr(w, "target_species", -1) >= 0:
            self.set_neutral_target(w.target_species)
        for k, s in enumerate(w.species):   # NEXT-2: part of the configuration, set before any load or restart
            if getattr(s, "recycle_to", -1) >= 0:
                self.set_recycling(k, s.recycle_to, s.recycle_vth)

    def close(self):
        if getattr(self, "h", None):
            self.lib.bit1_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- bit1_load_particles ----------------------------------------------------------------
    def load_particles(self, x, vx, vy, vz, sp, pid=None):
        """numpy arrays (HOST) or torch CUDA tensors (DEVICE), all of one kind."""
        on_device = not isinstance(x, np.ndarray) and getattr(x, "is_cuda", False)
        if not on_device:
            x, vx, vy, vz = _f8(x), _f8(vx), _f8(vy), _f8(vz)
            sp = np.ascontiguousarray(np.asarray(sp, dtype=np.uint8))
            if pid is not None:
                pid = np.ascontiguousarray(np.asarray(pid, dtype=np.uint32))
        else:
            self._torch.cuda.current_stream().synchronize()
        n = int(x.shape[0])
        _check(self.lib.bit1_load_particles(self.h, n, _ptr(x), _ptr(vx), _ptr(vy), _ptr(vz), _ptr(sp), _ptr(pid),
                                            int(on_device)), "bit1_load_particles")

    def load(self):
        w = self.w
        self.load_particles(w.x, w.vx, w.vy, w.vz, w.sp)

    # -- bit1_step / bit1_sync --------------------------------------------------------------
    def step(self, n: int = 1):
        _check(self.lib.bit1_step(self.h, int(n)), "bit1_step")

    def sync(self, check_flags: bool = True):
        s = self.lib.bit1_sync(self.h)
        if s == ERR_DEVICE_FLAG and not check_flags:
            return
        _check(s, "bit1_sync")

    # -- getters -----------------------------------------------------------------------------
    def get_count(self):
        n, st = C.c_uint64(), C.c_uint64()
        per = (C.c_uint64 * MAX_SPECIES)()
        _check(self.lib.bit1_get_count(self.h, C.byref(n), C.byref(st), per), "bit1_get_count")
        return int(n.value), int(st.value), np.array(per[: self.ns], dtype=np.uint64)

    def n_live(self):
        n, st = C.c_uint64(), C.c_uint64()
        _check(self.lib.bit1_get_count(self.h, C.byref(n), C.byref(st), None), "bit1_get_count")
        return int(n.value)

    def get_rho(self, si: bool = False):
        r = np.zeros(self.ng, np.int64)
        rs = np.zeros(self.ng) if si else None
        _check(self.lib.bit1_get_rho(self.h, r.ctypes.data, rs.ctypes.data if si else None), "bit1_get_rho")
        return (r, rs) if si else r

    def get_phi(self):
        a = np.zeros(self.nc + 1)
        _check(self.lib.bit1_get_phi(self.h, a.ctypes.data), "bit1_get_phi")
        return a

    def get_E(self):
        a = np.zeros(self.nc + 1)
        _check(self.lib.bit1_get_E(self.h, a.ctypes.data), "bit1_get_E")
        return a

    def get_dens(self):
        a = np.zeros((self.ns, self.ng), np.int64)
        _check(self.lib.bit1_get_dens(self.h, a.ctypes.data), "bit1_get_dens")
        return a

    def get_moments(self, density: bool = False):
        m = bit1_moments()
        dens = None
        if density:
            dens = np.zeros((self.ns, self.ng))
            for k in range(self.ns):
                m.density[k] = dens[k].ctypes.data_as(c_f64p)
        _check(self.lib.bit1_get_moments(self.h, C.byref(m)), "bit1_get_moments")
        ns = self.ns
        out = dict(step=int(m.step), n_live=int(m.n_live), count=np.array(m.count[:ns], np.uint64),
                   kinetic_J=np.array(m.kinetic_J[:ns]), px=np.array(m.px[:ns]), field_J=float(m.field_J),
                   wall_count=np.array([list(m.wall_count[0][:ns]), list(m.wall_count[1][:ns])], np.uint64),
                   wall_charge=np.array(m.wall_charge_fixed[:], np.int64), rho_total=int(m.rho_total_fixed),
                   flags=int(m.flags), next_pid=int(m.next_pid), nu_overflow=int(m.nu_overflow),
                   dir_fallback=int(m.dir_fallback), escape=int(m.escape), births=int(m.births),
                   reinject=int(m.reinject), candidates=np.array(m.candidates[:ns], np.uint64),
                   events=np.array([list(m.events[k][:]) for k in range(ns)], np.uint64),
                   far_movers=int(m.far_movers), max_far_movers_per_step=int(m.max_far_movers_per_step),
                   recycled=int(m.recycled), general_steps=int(m.general_steps), window_radius=int(m.window_radius),
                   check_failures=int(m.check_failures), check_line=int(m.check_line),
                   check_index=int(m.check_index), check_limit=int(m.check_limit))
        if density:
            out["density"] = dens
        return out

    def get_particles(self, cell_start: bool = True):
        n = self.n_live()
        d = dict(x=np.zeros(n), vx=np.zeros(n), vy=np.zeros(n), vz=np.zeros(n), cell=np.zeros(n, np.int32),
                 pid=np.zeros(n, np.uint32), sp=np.zeros(n, np.uint8))
        cs = np.zeros(self.nc + 1, np.int64) if cell_start else None
        _check(self.lib.bit1_get_particles(self.h, d["x"].ctypes.data, d["vx"].ctypes.data, d["vy"].ctypes.data,
                                           d["vz"].ctypes.data, d["cell"].ctypes.data, d["pid"].ctypes.data,
                                           d["sp"].ctypes.data, cs.ctypes.data if cell_start else None),
               "bit1_get_particles")
        if cell_start:
            d["cell_start"] = cs
        return d

    def set_neutral_target(self, species: int):
        _check(self.lib.bit1_set_neutral_target(self.h, int(species)), "bit1_set_neutral_target")

    def set_recycling(self, species: int, to_species: int, vth: float):
        _check(self.lib.bit1_set_recycling(self.h, int(species), int(to_species), float(vth)), "bit1_set_recycling")

    # -- NEXT-1: density smoothing, time-averaged diagnostics ----------------------------------
    def set_smoothing(self, passes: int):
        _check(self.lib.bit1_set_smoothing(self.h, int(passes)), "bit1_set_smoothing")

    def get_rho_smoothed(self):
        r = np.zeros(self.ng, np.int64)
        _check(self.lib.bit1_get_rho_smoothed(self.h, r.ctypes.data), "bit1_get_rho_smoothed")
        return r

    def set_averaging(self, window: int, interval: int):
        _check(self.lib.bit1_set_averaging(self.h, int(window), int(interval)), "bit1_set_averaging")

    def get_average(self):
        """Latest latched window: (dens_sum[ns, ng] int64, phi_sum[nc+1], count, step)."""
        d = np.zeros((self.ns, self.ng), np.int64)
        f = np.zeros(self.nc + 1)
        cnt, st = C.c_uint64(), C.c_uint64()
        _check(self.lib.bit1_get_average(self.h, d.ctypes.data, f.ctypes.data, C.byref(cnt), C.byref(st)),
               "bit1_get_average")
        return d, f, int(cnt.value), int(st.value)

    def set_E(self, E, freeze_field: bool = True):
        E = _f8(E)
        assert E.shape[0] == self.nc + 1
        _check(self.lib.bit1_set_E(self.h, E.ctypes.data, int(freeze_field)), "bit1_set_E")

    def set_step(self, step: int):
        _check(self.lib.bit1_set_step(self.h, int(step)), "bit1_set_step")

    # -- checkpoint / restart ------------------------------------------------------------------
    def checkpoint_size(self) -> int:
        return int(self.lib.bit1_checkpoint_size(self.h))

    def checkpoint(self, pinned):
        """pinned: torch uint8 CPU tensor in pinned memory, >= checkpoint_size() bytes."""
        written = C.c_size_t()
        _check(self.lib.bit1_checkpoint(self.h, pinned.data_ptr(), pinned.numel(), C.byref(written)),
               "bit1_checkpoint")
        return int(written.value)

    def checkpoint_wait(self):
        _check(self.lib.bit1_checkpoint_wait(self.h), "bit1_checkpoint_wait")

    def restart(self, blob):
        _check(self.lib.bit1_restart(self.h, blob.data_ptr(), blob.numel()), "bit1_restart")

    def export_species(self, species: int):
        """One species in the paper's checkpoint layout: dict(counts[nc] int64, x, vx, vy, vz, pid) in cell order."""
        n = C.c_uint64()
        counts = np.zeros(self.nc, np.int64)
        _check(self.lib.bit1_export_species(self.h, int(species), 0, C.byref(n), counts.ctypes.data, None, None, None,
                                            None, None), "bit1_export_species (size query)")
        m = int(n.value)
        d = dict(x=np.zeros(m), vx=np.zeros(m), vy=np.zeros(m), vz=np.zeros(m), pid=np.zeros(m, np.uint32))
        _check(self.lib.bit1_export_species(self.h, int(species), m, C.byref(n), counts.ctypes.data, d["x"].ctypes.data,
                                            d["vx"].ctypes.data, d["vy"].ctypes.data, d["vz"].ctypes.data,
                                            d["pid"].ctypes.data), "bit1_export_species")
        d["counts"] = counts
        return d

    # -- streaming checkpoints (NEXT-4) ------------------------------------------------------------
    def stream_slot_size(self) -> int:
        return int(self.lib.bit1_stream_slot_size(self.h))

    def stream_open(self, ring, nslots: int):
        """ring: pinned torch uint8 CPU tensor of nslots equal slots (256-byte aligned, slot size a multiple of 256)."""
        self._ring = ring
        self._slot_bytes = ring.numel() // nslots
        _check(self.lib.bit1_stream_open(self.h, ring.data_ptr(), self._slot_bytes, int(nslots)), "bit1_stream_open")

    def stream_publish(self) -> int:
        seq = C.c_uint64()
        _check(self.lib.bit1_stream_publish(self.h, C.byref(seq)), "bit1_stream_publish")
        return int(seq.value)

    def stream_acquire(self, after_seq: int = 0):
        """Newest complete snapshot with a sequence number > after_seq, or None.  Returns (seq, snapshot): step,
        n_total and per species a dict(counts[nc] int32, x, vx, vy, vz, pid) of numpy VIEWS of the pinned slot, valid
        until stream_release(seq)."""
        slot, seq = C.c_void_p(), C.c_uint64()
        st = self.lib.bit1_stream_acquire(self.h, int(after_seq), C.byref(slot), C.byref(seq))
        if st == ERR_STATE:
            return None
        _check(st, "bit1_stream_acquire")
        hd = bit1_stream_header.from_address(slot.value)
        assert hd.magic == b"BIT1STRM" and hd.seq == hd.seq_begin == seq.value

        def view(off, n, dt):
            nbytes = n * np.dtype(dt).itemsize
            buf = (C.c_char * nbytes).from_address(slot.value + off)
            return np.frombuffer(buf, dtype=dt, count=n)

        sp = []
        for s in range(hd.ns):
            n = int(hd.count[s])
            sp.append(dict(counts=view(hd.off_counts[s], hd.nc, np.int32), x=view(hd.off_x[s], n, np.float64),
                           vx=view(hd.off_vx[s], n, np.float64), vy=view(hd.off_vy[s], n, np.float64),
                           vz=view(hd.off_vz[s], n, np.float64), pid=view(hd.off_pid[s], n, np.uint32)))
        return int(seq.value), dict(step=int(hd.step), n_total=int(hd.n_total), bytes=int(hd.bytes), species=sp)

    def stream_release(self, seq: int):
        _check(self.lib.bit1_stream_release(self.h, int(seq)), "bit1_stream_release")

    def stream_close(self):
        _check(self.lib.bit1_stream_close(self.h), "bit1_stream_close")

    def profile(self, enable: bool = True):
        _check(self.lib.bit1_profile(self.h, int(enable)), "bit1_profile")

    def get_profile(self):
        ms = (C.c_double * 4)()
        steps = C.c_uint64()
        _check(self.lib.bit1_get_profile(self.h, C.byref(ms), C.byref(steps)), "bit1_get_profile")
        return dict(zip(("pass_a", "mid", "pass_b", "field"), [float(v) for v in ms])), int(steps.value)

    def check_selftest(self):
        _check(self.lib.bit1_check_selftest(self.h), "bit1_check_selftest")

    def launch_count(self) -> int:
        return int(self.lib.bit1_launch_count(self.h))
