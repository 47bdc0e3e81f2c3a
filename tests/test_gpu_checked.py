"""The parity cases again on libbit1_checked.so: the same sources built with -DBIT1_CHECKED, in which every index the
step kernels compute from particle data (shared-memory histogram / window / deposit slots, scatter destinations,
side-list slots, banded-row offsets, cell indices, radix destinations) is compared with its bound before use
(csrc/common.cuh BIT1_CHECK).  compute-sanitizer is closed on this GPU pool (profiles/r2_sanitizer.md), so these
checks, the oracle comparison and the two-run determinism test are the memory-safety evidence.  Each case must match
the oracle bit for bit AND record zero failed checks."""
import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import assert_state_equal

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def checked():
    from paper_2606_28534_b200 import binding, build

    lib = binding.load_library(build.build(checked=True))
    assert lib.bit1_build_is_checked() == 1
    assert binding.load_library().bit1_build_is_checked() == 0
    return lib


def _run(lib, w, chunks, **kw):
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    g = Bit1(w, lib=lib, **kw)
    g.load()
    o = Oracle(w)
    for c in chunks:
        g.step(c)
        o.step(c)
    g.sync(check_flags=False)
    m = g.get_moments()
    assert m["check_failures"] == 0, (f"index check failed at line {m['check_line']}: index {m['check_index']} "
                                      f"against bound {m['check_limit']} ({m['check_failures']} failures)")
    assert assert_state_equal(g, o, where="checked build")
    return g, m


def test_the_checks_fire_on_a_bad_index(checked):
    from paper_2606_28534_b200.binding import Bit1, Bit1Error, ERR_STATE

    w = W.make_config(1, scale=1 / 16)
    g = Bit1(w, lib=checked)
    g.load()
    g.check_selftest()            # an out-of-range index is caught, recorded and redirected
    assert g.get_moments()["check_failures"] == 0   # the self-test clears its own record
    g.close()
    h = Bit1(w)
    h.load()
    with pytest.raises(Bit1Error) as e:
        h.check_selftest()        # the shipped library has no checks compiled in
    assert e.value.status == ERR_STATE
    h.close()


@pytest.mark.parametrize("cfg,scale,kw,bit1_kw", [
    (1, 1 / 4, {}, {}),
    (2, 1 / 32, dict(pair_source=True, recycle=True), {}),
    (3, 1 / 128, dict(n0_scale=300.0, pair_source=True), {}),
    (3, 1 / 128, dict(n0_scale=300.0), dict(direct_launch=True)),
    (4, 1 / 1024, dict(n0_scale=100.0), dict(window_radius=0)),
    (5, 1 / 4096, dict(n0_scale=100.0, recycle=True), dict(window_radius=60)),
    (3, 1 / 128, dict(n0_scale=300.0, pair_source=True, recycle=True), dict(side_list_capacity=16)),   # general path
])
def test_parity_cases_pass_every_index_check(checked, cfg, scale, kw, bit1_kw):
    w = W.make_config(cfg, scale=scale, **kw)
    g, m = _run(checked, w, (1, 7, 12), **bit1_kw)
    g.close()


@pytest.mark.parametrize("boost,bit1_kw", [(8.0, dict(window_radius_max=40)), (40.0, {}),
                                           (10.0, dict(window_radius=0, side_list_capacity=1 << 20))])
def test_hot_plasmas_long_side_lists_and_wide_windows_pass_every_index_check(checked, boost, bit1_kw):
    w = W.make_config(3, scale=1 / 64, n0_scale=2000.0, pair_source=True, recycle=True)
    for k in ("vx", "vy", "vz"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k) * boost))
    g, m = _run(checked, w, (2, 5), **bit1_kw)
    g.close()


def test_sparse_tiles_and_a_single_dense_cell_pass_every_index_check(checked):
    rng = np.random.default_rng(5)
    w = W.make_config(2, scale=1 / 4)   # 1024 cells, ~1.5 particles per cell: tiles wider than the window
    sel = np.sort(rng.choice(w.n, size=1500, replace=False))
    for k in ("x", "vx", "vy", "vz", "sp"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k)[sel]))
    g, m = _run(checked, w, (3, 4))
    assert m["far_movers"] > 0
    g.close()
    w = W.make_config(2, scale=1 / 64)
    n = 6000
    for k in ("vx", "vy", "vz", "sp"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k)[:n]))
    w.x = np.ascontiguousarray((17 + rng.random(n)) * w.dx)
    g, m = _run(checked, w, (4,))
    g.close()


def test_mid_size_and_million_cell_grids_pass_every_index_check(checked):
    w = W.make_config(4, scale=1 / 16, n0_scale=30.0)     # 1.25e7 particles: stages reloaded dozens of times
    g, m = _run(checked, w, (3,))
    g.close()
    w = W.make_config(5, ppc_scale=1 / 120, n0_scale=100.0)   # 1 048 576 cells, 8.3e6 particles
    g, m = _run(checked, w, (2,))
    g.close()


def test_restart_and_streaming_on_the_checked_build(checked):
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    w = W.make_config(3, scale=1 / 128, n0_scale=200.0, pair_source=True)
    g = Bit1(w, lib=checked, checkpoint_staging=True)
    g.load()
    g.step(6)
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    nbytes = g.checkpoint(blob)
    g.step(3)
    g.checkpoint_wait()
    slot = (g.stream_slot_size() + 255) // 256 * 256
    ring = torch.empty(2 * slot, dtype=torch.uint8).pin_memory()
    g.stream_open(ring, 2)
    g.stream_publish()
    g.checkpoint_wait()
    seq, snap = g.stream_acquire(0)
    assert snap["step"] == 9 and snap["n_total"] == g.n_live()
    g.stream_release(seq)
    g.stream_close()
    assert g.get_moments()["check_failures"] == 0
    g.close()
    h = Bit1(w, lib=checked)
    h.restart(blob[:nbytes])
    h.step(5)
    h.sync(check_flags=False)
    o = Oracle(w)
    o.step(11)
    assert h.get_moments()["check_failures"] == 0
    assert assert_state_equal(h, o, where="checked build, restarted")
    h.close()
