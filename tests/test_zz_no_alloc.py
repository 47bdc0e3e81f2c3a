"""bit1_field_solve_static: the field solve for callers that may not allocate GPU memory.

Who needs it: code that lives inside somebody else's program -- a plug-in whose host hands out device memory from its
own pool, a callback that runs while that pool is locked, a job whose device-memory budget was fixed at start-up.  Such
a caller cannot cudaMalloc the workspace every other libbit1 call works out of.  This entry point therefore keeps its
temporaries in an array built into libbit1.so (hence the ceiling of BIT1_FIELD_STATIC_MAX_CELLS cells) and allocates
nothing.

What is checked: phi and E from the new entry point against the ordinary path (a context: bit1_set_smoothing,
bit1_step, bit1_get_rho / bit1_get_phi / bit1_get_E) on the same rho.  The solve is exact integer arithmetic followed by
one conversion and one multiplication per node, and the other field tests of this suite demand identical bits, so this
one does too.  Every case makes two (or more) calls in a row on one stream without waiting in between, on different
grids, so that a call which relied on the built-in array being clean -- or which looked at what the previous call left
there -- would fail.

The file name sorts last on purpose: pytest -x stops at the first failure, and a problem here should not hide the
results of the older tests.  The tests neither need nor disturb anything the other files set up; they pass in a fresh
process and at the end of the whole run alike."""
import ctypes

import numpy as np
import pytest

from paper_2606_28534_b200 import binding
from paper_2606_28534_b200 import workloads as W


def _reference(w, passes, steps):
    """rho, phi, E of the ordinary path after `steps` steps with `passes` smoothing passes."""
    from paper_2606_28534_b200.binding import Bit1

    g = Bit1(w)
    g.set_smoothing(passes)
    g.load()
    g.step(steps)
    g.sync(check_flags=False)
    rho, phi, E = g.get_rho(), g.get_phi(), g.get_E()
    g.close()
    assert np.any(rho != 0), "a rho of zeros would prove nothing"
    return dict(w=w, passes=passes, rho=rho, phi=phi, E=E)


def _enqueue_static(ref, stream=None):
    """One call of the new entry point on device copies of ref's rho; returns the output tensors (not yet waited for)."""
    import torch

    w = ref["w"]
    rho_d = torch.from_numpy(ref["rho"]).cuda()
    phi_d = torch.full((w.nc + 1,), float("nan"), dtype=torch.float64, device="cuda")
    E_d = torch.full((w.nc + 1,), float("nan"), dtype=torch.float64, device="cuda")
    binding.field_solve_static(rho_d, phi_d, E_d, w.nc, w.bc, w.dx, w.area, ref["passes"], stream=stream)
    return rho_d, phi_d, E_d


def _assert_same(ref, out, where):
    rho_d, phi_d, E_d = out
    assert np.array_equal(rho_d.cpu().numpy(), ref["rho"]), f"{where}: the input was written to"
    phi, E = phi_d.cpu().numpy(), E_d.cpu().numpy()
    assert np.array_equal(phi, ref["phi"]), f"{where}: phi differs at {np.flatnonzero(phi != ref['phi'])[:5]}"
    assert np.array_equal(E, ref["E"]), f"{where}: E differs at {np.flatnonzero(E != ref['E'])[:5]}"


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_context_path():
    import torch

    # walls, B field, collisions: 4096 cells -> five CTAs meeting at grid barriers; two smoothing passes use both arrays
    a = _reference(W.make_config(3, scale=1 / 4, n0_scale=100.0), passes=2, steps=12)
    # periodic, independently loaded charges (rho != 0 from the start), 3072 cells, one pass
    b = _reference(W.make_config(1, scale=3, quiet=False), passes=1, steps=7)
    # the one-CTA path (<= 1025 nodes), no smoothing: reads rho directly
    c = _reference(W.make_config(1, quiet=False), passes=0, steps=5)
    assert a["w"].bc == 1 and b["w"].bc == 0 and a["w"].nc == 4096 and b["w"].nc == 3072 and c["w"].nc == 1024
    torch.cuda.synchronize()

    outs = [(_enqueue_static(r), r, name) for r, name in ((a, "first call"), (b, "second call, smaller grid"))]
    torch.cuda.synchronize()
    for out, r, name in outs:
        _assert_same(r, out, name)

    # again in another order, back to back, with device memory watched: the calls themselves allocate nothing
    # (the tensors are made beforehand; the first round above has already loaded the kernel's module)
    pre = [(r, torch.from_numpy(r["rho"]).cuda(), torch.empty(r["w"].nc + 1, dtype=torch.float64, device="cuda"),
            torch.empty(r["w"].nc + 1, dtype=torch.float64, device="cuda")) for r in (c, a, b, a, c)]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for r, rho_d, phi_d, E_d in pre:
        w = r["w"]
        binding.field_solve_static(rho_d, phi_d, E_d, w.nc, w.bc, w.dx, w.area, r["passes"])
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    for k, (r, rho_d, phi_d, E_d) in enumerate(pre):
        _assert_same(r, (rho_d, phi_d, E_d), f"round two, call {k}")
    assert free_after >= free_before, f"device memory in use grew by {free_before - free_after} bytes across the calls"


@pytest.mark.gpu
def test_the_largest_grid_it_accepts_twice_in_a_row():
    import torch

    # BIT1_FIELD_STATIC_MAX_CELLS cells with walls: nc + 1 nodes, every byte of both smoothing arrays in use (8 passes),
    # the cooperative grid at its cap
    big = _reference(W.make_config(5, ppc_scale=1 / 60, n0_scale=100.0), passes=8, steps=2)
    assert big["w"].nc == binding.FIELD_STATIC_MAX_CELLS and big["w"].bc == 1
    small = _reference(W.make_config(2, scale=1 / 2), passes=3, steps=20)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()          # a stream of the caller's choosing, not torch's current one
    side.wait_stream(torch.cuda.current_stream())
    o1 = _enqueue_static(big, stream=side)
    o2 = _enqueue_static(small, stream=side)   # leaves most of the big call's temporaries in place
    o3 = _enqueue_static(big, stream=side)
    side.synchronize()
    _assert_same(big, o1, "largest grid, first call")
    _assert_same(small, o2, "small grid after the largest")
    _assert_same(big, o3, "largest grid again")


def test_refusals_come_before_any_gpu_work():
    """Argument checks need no device: nothing is dereferenced or launched when a call is refused."""
    L = binding.load_library()
    fake = ctypes.c_void_p(4096)   # never touched
    ok_args = (fake, fake, fake, 1024, 1, 1e-5, 1.0, 0, None)

    def call(**kw):
        names = ("rho", "phi", "E", "nc", "bc", "dx", "area", "passes", "stream")
        a = dict(zip(names, ok_args))
        a.update(kw)
        return L.bit1_field_solve_static(*[a[n] for n in names])

    assert call(nc=binding.FIELD_STATIC_MAX_CELLS + 1) == binding.ERR_STATIC_LIMIT
    assert call(nc=1 << 27, bc=0) == binding.ERR_STATIC_LIMIT
    msg = L.bit1_error_string(binding.ERR_STATIC_LIMIT).decode()
    assert "BIT1_FIELD_STATIC_MAX_CELLS" in msg and str(binding.FIELD_STATIC_MAX_CELLS) in msg
    for bad in (dict(rho=None), dict(phi=None), dict(E=None), dict(nc=1), dict(bc=2), dict(dx=0.0), dict(area=-1.0),
                dict(dx=float("nan")), dict(passes=-1), dict(passes=9)):
        assert call(**bad) == binding.ERR_INVALID_ARG, bad
