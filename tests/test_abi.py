"""The C-ABI library loads and exports every symbol include/bit1.h declares (no compute calls)."""
import ctypes
import os
import re

from paper_2606_28534_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "bit1.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bit1_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    names = declared_symbols()
    assert len(names) >= 20 and "bit1_step" in names and "bit1_restart" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/bit1.h but not exported"


def test_binding_declares_the_same_entry_points():
    L = binding.load_library()
    for n in declared_symbols():
        fn = getattr(L, n)
        assert fn.argtypes is not None, f"binding.py does not declare {n}"


def test_host_side_argument_checks_need_no_gpu():
    L = binding.load_library()
    g = binding.bit1_grid(1, 1, 1e-5, 1.0, 0, 0, 0)  # nc < 2
    o = binding.bit1_options()
    o.capacity = 1000
    assert L.bit1_workspace_size(ctypes.byref(g), 2, ctypes.byref(o)) == 0
    g = binding.bit1_grid(1024, 1, 1e-5, 1.0, 0, 0, 0)
    o.capacity = 100000
    a = L.bit1_workspace_size(ctypes.byref(g), 2, ctypes.byref(o))
    o.checkpoint_staging = 1
    b = L.bit1_workspace_size(ctypes.byref(g), 2, ctypes.byref(o))
    assert a > 2 * 41 * 100000 and b >= a
    o.window_radius_max = 60
    assert L.bit1_workspace_size(ctypes.byref(g), 2, ctypes.byref(o)) > b      # wider rows of the banded arrays
    o.window_radius_max = 61
    assert L.bit1_workspace_size(ctypes.byref(g), 2, ctypes.byref(o)) == 0     # beyond the shared-memory window
    o.window_radius_max = 0
    o.side_list_capacity = 8
    assert L.bit1_workspace_size(ctypes.byref(g), 2, ctypes.byref(o)) == 0
    o.side_list_capacity = 0
    assert L.bit1_workspace_size(ctypes.byref(g), 9, ctypes.byref(o)) == 0  # too many species
    assert L.bit1_workspace_size(ctypes.byref(g), 2, None) == 0
    assert L.bit1_error_string(7) == b"sticky device flag set"
    h = ctypes.c_void_p()
    assert L.bit1_create(None, None, 0, 0.0, None, ctypes.byref(h)) == binding.ERR_INVALID_ARG
    assert L.bit1_step(None, 1) == binding.ERR_INVALID_ARG


def test_struct_sizes_match_the_header():
    # layout of the C structs as documented in include/bit1.h (natural alignment)
    assert ctypes.sizeof(binding.bit1_grid) == 48
    assert ctypes.sizeof(binding.bit1_species) == 64
    assert ctypes.sizeof(binding.bit1_options) == 8 * 8 + 3 * 8 + 8 + 8 + 8 + 8 + 8 + 8 + 8 + 4 * 4 + 8
