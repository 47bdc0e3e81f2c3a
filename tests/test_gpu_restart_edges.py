"""GPU tests beyond the plain parity cases: checkpoint/restart, determinism,
edge cases (empty input, capacity hit, window radius, degenerate tiles) and the error behaviour of the C ABI.
Everything goes through the C ABI (paper_2606_28534_b200.binding) and is compared with the CPU oracle."""
import os

import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import run_pair, assert_state_equal

pytestmark = pytest.mark.gpu


def _state(g):
    p = g.get_particles()
    p["rho"] = g.get_rho()
    p["dens"] = g.get_dens()
    p["E"] = g.get_E()
    p["phi"] = g.get_phi()
    m = g.get_moments()
    p["wall_count"], p["wall_charge"] = m["wall_count"], m["wall_charge"]
    p["scalars"] = np.array([m["step"], m["next_pid"], m["births"], m["reinject"], m["flags"], m["rho_total"]],
                            dtype=np.int64)
    p["events"], p["candidates"] = m["events"], m["candidates"]
    return p


def _assert_identical(a, b, where):
    assert a.keys() == b.keys()
    for k in a:
        assert np.array_equal(a[k], b[k]), f"{where}: {k} differs"


@pytest.mark.parametrize("staging", [False, True])
@pytest.mark.parametrize("cfg,scale,kw", [
    (2, 1 / 32, dict(pair_source=True)),
    (3, 1 / 128, dict(n0_scale=200.0)),
    (5, 1 / 8192, dict(n0_scale=200.0)),
])
def test_checkpoint_restart_is_bit_identical(cfg, scale, kw, staging):
    """run 0 -> m  ==  run 0 -> k, checkpoint, (keep stepping), restart from the blob, k -> m; also == oracle."""
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    k, m = 7, 19
    w = W.make_config(cfg, scale=scale, **kw)
    ref = Bit1(w)
    ref.load()
    ref.step(m)
    ref.sync(check_flags=False)
    want = _state(ref)
    ref.close()

    g = Bit1(w, checkpoint_staging=staging)
    g.load()
    g.step(k)
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    written = g.checkpoint(blob)
    assert 0 < written <= g.checkpoint_size()   # the blob holds the live particles only, the size call says the worst case
    g.step(5)  # the snapshot must not see these steps (they overlap the D2H copy when staging is on)
    g.checkpoint_wait()
    g.sync(check_flags=False)
    g.close()

    h = Bit1(w, checkpoint_staging=staging)  # a fresh context, as after a crash
    h.restart(blob[:written])
    assert h.get_moments()["step"] == k
    h.step(m - k)
    h.sync(check_flags=False)
    _assert_identical(_state(h), want, f"c{cfg} restart staging={staging}")

    o = Oracle(w)
    o.step(m)
    assert assert_state_equal(h, o, where=f"c{cfg} restarted run vs oracle")
    h.close()


def test_restart_rejects_a_blob_of_another_configuration():
    import torch
    from paper_2606_28534_b200.binding import Bit1, Bit1Error, ERR_CHECKPOINT

    w = W.make_config(2, scale=1 / 64)
    g = Bit1(w)
    g.load()
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    g.checkpoint(blob)
    g.checkpoint_wait()
    g.close()
    w2 = W.make_config(2, scale=1 / 64, lib_seed=99)  # same sizes, other seed -> other config hash
    h = Bit1(w2)
    with pytest.raises(Bit1Error) as e:
        h.restart(blob)
    assert e.value.status == ERR_CHECKPOINT
    bad = blob.clone()
    bad[0] = 0  # magic
    with pytest.raises(Bit1Error):
        Bit1(w).restart(bad)
    h.close()


def test_restart_refuses_a_blob_whose_body_was_tampered_with_and_create_refuses_a_bad_source_interval():
    """The blob's header and hash vouch for the configuration only: a species tag that does not exist, a position
    outside the domain and positions out of cell order are caught on the device before anything indexes by them
    (BIT1_ERR_CHECKPOINT, no device fault; the context can be loaded again).  bit1_create refuses re-injection
    intervals that are empty or reach outside [0, L) when a species re-injects."""
    import torch
    from paper_2606_28534_b200.binding import Bit1, Bit1Error, ERR_CHECKPOINT, ERR_INVALID_ARG

    w = W.make_config(2, scale=1 / 64)
    g = Bit1(w)
    g.load()
    g.step(3)
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    written = g.checkpoint(blob)
    g.checkpoint_wait()
    n = g.n_live()
    x = g.get_particles()["x"]
    raw = blob.numpy()
    sp_off = written - (n + 255) // 256 * 256          # the species tags are the blob's last section
    x_off = raw[:written].tobytes().find(x[:4].tobytes())
    assert x_off > 0 and x_off % 256 == 0, "the positions' section was not found"
    for what in ("species", "position", "order"):
        bad = blob.clone()
        b = bad.numpy()
        if what == "species":
            b[sp_off + 3] = 200
        elif what == "position":
            b[x_off + 8 * 5: x_off + 8 * 6] = np.frombuffer(np.float64(-1.0).tobytes(), np.uint8)
        else:   # the first and the last particle change places: no longer sorted by cell
            first = b[x_off: x_off + 8].copy()
            b[x_off: x_off + 8] = b[x_off + 8 * (n - 1): x_off + 8 * n]
            b[x_off + 8 * (n - 1): x_off + 8 * n] = first
        with pytest.raises(Bit1Error) as e:
            g.restart(bad)
        assert e.value.status == ERR_CHECKPOINT, what
    g.restart(blob)   # the untouched blob still restarts, and the run goes on
    g.step(2)
    g.sync()
    g.close()
    L = w.nc * w.dx
    for lo, hi in ((0.5 * L, 0.5 * L), (0.75 * L, 0.25 * L), (-0.1 * L, 0.5 * L), (0.5 * L, 1.5 * L)):
        w.src_lo, w.src_hi = lo, hi
        with pytest.raises(Bit1Error) as e:
            Bit1(w)
        assert e.value.status == ERR_INVALID_ARG, (lo, hi)


def test_two_runs_give_identical_bits():
    w = W.make_config(3, scale=1 / 64, n0_scale=100.0)
    a, _ = None, None
    from paper_2606_28534_b200.binding import Bit1

    states = []
    for _ in range(2):
        g = Bit1(w)
        g.load()
        g.step(25)
        g.sync(check_flags=False)
        states.append(_state(g))
        g.close()
    _assert_identical(states[0], states[1], "determinism")


def test_empty_input_steps_and_reports_zero():
    from paper_2606_28534_b200.binding import Bit1

    w = W.make_config(2, scale=1 / 64)
    g = Bit1(w)
    e = np.zeros(0)
    g.load_particles(e, e, e, e, np.zeros(0, np.uint8))
    g.step(3)
    g.sync()
    assert g.n_live() == 0
    assert not g.get_rho().any() and not g.get_E().any() and not g.get_phi().any()
    m = g.get_moments()
    assert m["step"] == 3 and m["n_live"] == 0 and m["flags"] == 0
    g.close()


@pytest.mark.parametrize("n", [1, 31, 1023, 1024, 1025, 2049])
def test_ragged_and_single_tile_sizes(n):
    """Particle counts around the tile size (1024): one particle, one warp minus one, exactly one tile, one
    tile plus a one-particle tail."""
    w0 = W.make_config(3, scale=1 / 256, n0_scale=300.0)
    idx = np.random.default_rng(5).choice(w0.n, size=n, replace=False)
    idx.sort()
    for k in ("x", "vx", "vy", "vz", "sp"):
        setattr(w0, k, np.ascontiguousarray(getattr(w0, k)[idx]))
    g, o = run_pair(w0, 5)
    assert assert_state_equal(g, o, where=f"n={n}")
    g.close()


def test_all_particles_in_one_cell_and_sparse_cells():
    """Degenerate tiles: every particle in one cell (a cell spanning many tiles), and a plasma so thin that a
    tile spans more cells than the shared-memory window holds (the rest goes through the side list)."""
    w = W.make_config(2, scale=1 / 64)
    n = 6000
    rng = np.random.default_rng(11)
    L = w.nc * w.dx
    for k in ("vx", "vy", "vz", "sp"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k)[:n]))
    w.x = np.ascontiguousarray((17 + rng.random(n)) * w.dx)  # all in cell 17
    g, o = run_pair(w, 4)
    assert assert_state_equal(g, o, where="one cell")
    g.close()
    w = W.make_config(2, scale=1 / 4)  # 1024 cells
    n = 1500  # ~1.5 particles per cell: a 1024-particle tile spans ~700 cells > window capacity
    sel = np.sort(rng.choice(w.n, size=n, replace=False))
    for k in ("x", "vx", "vy", "vz", "sp"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k)[sel]))
    g, o = run_pair(w, 3)
    assert assert_state_equal(g, o, where="sparse cells")
    assert g.get_moments()["far_movers"] > 0
    g.close()


@pytest.mark.parametrize("bc_cfg", [1, 2])
def test_deposit_at_nodes_cell_edges_and_the_last_representable_position(bc_cfg):
    """The CIC split at its edges (SURVEY 8(c) "D": F = 0 for f <= 0, 2^32 - 1 for f >= 1, else trunc(f 2^32)): particles
    exactly on nodes, one ulp either side of them, at 0, and at the last doubles below L, where x * inv_dx rounds up to nc,
    the cell clamps to nc - 1 and f becomes 1.  Cold particles in a field-free box: the load-time deposit and the fused
    deposit of the following steps see the same positions.  The CUDA path takes F with one saturating conversion."""
    w = W.make_config(bc_cfg, scale=1 / 16)
    # a cell size for which the last double below L times fl(1/dx) rounds up to nc: the clamp edge f = 1 exists
    for f in np.random.default_rng(3).random(2000):
        d = w.dx * (1.0 + 0.5 * f)
        if np.nextafter(w.nc * d, -np.inf) * (1.0 / d) >= w.nc:
            w.dx = float(d)
            break
    L = w.nc * w.dx
    assert np.nextafter(L, -np.inf) * (1.0 / w.dx) - (w.nc - 1) >= 1.0, "no clamp edge for this dx"
    if w.bc:
        w.src_lo, w.src_hi = 0.25 * L, 0.75 * L
    nodes = np.arange(w.nc, dtype=np.float64) * w.dx
    xs = [nodes, np.nextafter(nodes, np.inf), np.nextafter(nodes[1:], -np.inf), nodes + 0.5 * w.dx,
          nodes + w.dx * 2.0 ** -33, nodes + w.dx * (1.0 - 2.0 ** -33)]
    top = [L]
    for _ in range(64):
        top.append(np.nextafter(top[-1], -np.inf))
    xs.append(np.array(top[1:]))
    x = np.concatenate(xs)
    x = x[(x >= 0.0) & (x < L)]
    rng = np.random.default_rng(5)
    x = np.ascontiguousarray(rng.permutation(x))
    n = x.shape[0]
    w.x = x
    w.sp = np.ascontiguousarray((np.arange(n) % len(w.species)).astype(np.uint8))
    for k in ("vx", "vy", "vz"):
        setattr(w, k, np.zeros(n))
    for steps in (0, 2):
        g, o = run_pair(w, steps)
        assert assert_state_equal(g, o, where=f"deposit edges, bc {w.bc}, {steps} steps")
        g.close()


@pytest.mark.parametrize("cfg,scale,kw", [(1, 1 / 4, {}), (3, 1 / 256, dict(n0_scale=300.0, pair_source=True))])
def test_side_list_longer_than_one_cta_sorts_over_the_grid(cfg, scale, kw):
    """A plasma 40 times hotter than the grid was sized for: nearly every particle leaves its tile's window, so the
    side list (far movers and births) holds tens of thousands of entries and k_mid orders it with the grid-wide
    bitonic sort instead of one CTA's shared memory.  Same bits as the oracle, which has no such notion."""
    w = W.make_config(cfg, scale=scale, **kw)
    for k in ("vx", "vy", "vz"):
        setattr(w, k, np.ascontiguousarray(getattr(w, k) * 40.0))
    g, o = run_pair(w, 3)
    m = g.get_moments()
    assert m["max_far_movers_per_step"] > 4096, "the workload was meant to overflow one CTA's sort"
    assert assert_state_equal(g, o, where=f"c{cfg} hot plasma, long side list")
    g.close()


def test_capacity_hit_matches_oracle_and_raises_the_sticky_flag():
    """Ionisation births beyond capacity are dropped in (parent, kind) order and flag CAPACITY (reading R-W)."""
    from paper_2606_28534_b200.binding import Bit1Error, ERR_DEVICE_FLAG, FLAG_CAPACITY

    w = W.make_config(3, scale=1 / 256, n0_scale=3000.0, capacity_factor=1.0)
    w.capacity = w.n + 40
    g, o = run_pair(w, 12)
    assert o.flagword & FLAG_CAPACITY, "the workload was meant to run out of capacity"
    assert assert_state_equal(g, o, where="capacity")
    with pytest.raises(Bit1Error) as e:
        g.sync()
    assert e.value.status == ERR_DEVICE_FLAG
    g.close()


def test_particle_id_counter_wrap_matches_the_oracle_and_raises_the_flag():
    """Reading R-pid: ids are 32-bit on both sides.  Loaded with ids that end five short of 2^32, the ionisation births
    of the next steps take ids that wrap through 0: the CUDA path hands out the same ids as the oracle (which has the
    same counter and no flag) and raises BIT1_FLAG_PID_WRAP so that the shared random streams do not go unnoticed."""
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1, FLAG_PID_WRAP

    w = W.make_config(3, scale=1 / 256, n0_scale=300.0)
    pid = (np.arange(w.n, dtype=np.uint64) + (2 ** 32 - 5 - w.n)).astype(np.uint32)
    g = Bit1(w)
    g.load_particles(w.x, w.vx, w.vy, w.vz, w.sp, pid=pid)
    o = Oracle(w, load=False)
    o.load(w.x, w.vx, w.vy, w.vz, w.sp, pid=pid)
    g.step(3)
    o.step(3)
    g.sync(check_flags=False)
    m = g.get_moments()
    assert m["births"] > 5, "the workload was meant to create more births than ids were left"
    pg, po = g.get_particles(), o.particles()
    for k in ("pid", "sp", "cell", "x", "vx", "vy", "vz"):
        assert np.array_equal(pg[k], po[k]), k
    assert m["next_pid"] == o.next_pid and m["next_pid"] < 2 ** 31
    assert m["flags"] == (o.flagword | FLAG_PID_WRAP)
    assert np.array_equal(g.get_rho(), o.rho())
    g.close()


@pytest.mark.parametrize("R", [0, 2, 4, 17, 60])
def test_sort_window_radius_does_not_change_the_result(R):
    """Reading R-win: the radius only moves particles between the windowed path and the side list."""
    w = W.make_config(3, scale=1 / 128, n0_scale=200.0)
    g, o = run_pair(w, 10, window_radius=R)
    assert assert_state_equal(g, o, where=f"R={R}")
    assert g.get_moments()["window_radius"] == R
    g.close()
    w = W.make_config(1, scale=1 / 8)
    g, o = run_pair(w, 10, window_radius=R)
    assert assert_state_equal(g, o, where=f"R={R} periodic")
    g.close()


@pytest.mark.parametrize("boost,expect_wider", [(1.0, False), (12.0, True)])
def test_adaptive_window_radius_follows_the_displacements(boost, expect_wider):
    """The radius is chosen every step from the previous step's excess counts (k_mid): thermal particles at
    vth dt / dx = 0.2 keep it at 1; 12 x hotter ones (2.4 cells per step and sigma) widen it.  Same bits either way."""
    w = W.make_config(2, scale=1 / 16)
    for k in ("vx", "vy", "vz"):
        setattr(w, k, getattr(w, k) * boost)
    g, o = run_pair(w, 6, window_radius_max=40)
    assert assert_state_equal(g, o, where=f"adaptive radius, boost {boost}")
    m = g.get_moments()
    assert (m["window_radius"] > 4) == expect_wider, m["window_radius"]
    assert m["general_steps"] == 0
    g.close()


@pytest.mark.parametrize("cap,boost", [(16, 1.0), (64, 8.0), (2500, 40.0)])
def test_side_list_beyond_its_capacity_takes_the_general_path(cap, boost):
    """Reading R-side: a step whose far movers and births exceed the side-list capacity stalls on the device and is
    redone by the general path at the next call that waits; later steps are enqueued again.  Steps in uneven
    chunks, through graph replay and direct launches, with births, a pair source and recycling in play."""
    w = W.make_config(3, scale=1 / 128, n0_scale=500.0, pair_source=True, recycle=True)
    for k in ("vx", "vy", "vz"):
        setattr(w, k, getattr(w, k) * boost)
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    g = Bit1(w, side_list_capacity=cap, window_radius=1)
    g.load()
    o = Oracle(w)
    for chunk in (1, 9, 2, 12):
        g.step(chunk)
        o.step(chunk)
    g.sync(check_flags=False)
    m = g.get_moments()
    assert m["general_steps"] > 0, "the case was meant to overflow the side list"
    assert assert_state_equal(g, o, where=f"general path, capacity {cap}, boost {boost}")
    g.close()


def test_long_side_lists_are_radix_sorted_on_the_grid():
    """More than 2048 far movers + births per step: k_mid orders them with the grid-wide radix sort (and the births
    among them with a second one); pinned radius 0 and hot particles make nearly every particle a far mover."""
    w = W.make_config(3, scale=1 / 64, n0_scale=3000.0, pair_source=True, recycle=True)
    for k in ("vx", "vy", "vz"):
        setattr(w, k, getattr(w, k) * 10.0)
    g, o = run_pair(w, 5, window_radius=0, side_list_capacity=w.capacity)
    m = g.get_moments()
    assert m["max_far_movers_per_step"] > 20000 and m["general_steps"] == 0
    assert assert_state_equal(g, o, where="long side list")
    g.close()


def test_error_behaviour_of_the_c_abi():
    from paper_2606_28534_b200.binding import (Bit1, Bit1Error, ERR_CAPACITY, ERR_INVALID_ARG, ERR_RANGE,
                                               ERR_STATE)

    w = W.make_config(2, scale=1 / 64)
    g = Bit1(w)
    with pytest.raises(Bit1Error) as e:
        g.step(1)  # nothing loaded yet
    assert e.value.status == ERR_STATE
    big = np.zeros(w.capacity + 1)
    with pytest.raises(Bit1Error) as e:
        g.load_particles(big, big, big, big, np.zeros(big.shape[0], np.uint8))
    assert e.value.status == ERR_CAPACITY
    x = w.x.copy()
    x[5] = w.nc * w.dx * 1.5  # outside [0, L)
    with pytest.raises(Bit1Error) as e:
        g.load_particles(x, w.vx, w.vy, w.vz, w.sp)
    assert e.value.status == ERR_INVALID_ARG
    sp = w.sp.copy()
    sp[3] = 7  # no such species
    with pytest.raises(Bit1Error) as e:
        g.load_particles(w.x, w.vx, w.vy, w.vz, sp)
    assert e.value.status == ERR_INVALID_ARG
    g.load()  # the context is still usable
    g.step(2)
    g.sync()
    g.close()
    w.species[0].weight *= 1e9  # Q >= 2^31
    with pytest.raises(Bit1Error) as e:
        Bit1(w)
    assert e.value.status == ERR_RANGE


@pytest.mark.parametrize("cfg,scale,kw", [(2, 1 / 64, dict(pair_source=True)), (3, 1 / 256, dict(n0_scale=300.0))])
def test_heavy_macro_particles_take_the_64_bit_deposit_path(cfg, scale, kw):
    """Q_s >= 2^21 (here 400 x the workload's weight, with the cross-section area scaled alike so that the physics is
    unchanged): the shared-memory uint32 deposit counters could overflow, so the kernel deposits with 64-bit global
    reductions instead.  Same bits as the oracle."""
    w = W.make_config(cfg, scale=scale, **kw)
    w.area *= 400.0
    for s in w.species:
        s.weight *= 400.0
    g, o = run_pair(w, 25)
    assert int(o.Q().max()) >= 2**21
    assert assert_state_equal(g, o, where=f"c{cfg} heavy macro-particles")
    g.close()


def test_eight_species():
    """BIT1_MAX_SPECIES stored species with different masses, charges and weights in one periodic box."""
    rng = np.random.default_rng(8)
    nc, dx, n_per = 96, 2e-5, 900
    sp = []
    for k in range(8):
        q = (-1.0, 1.0, 0.0, 2.0)[k % 4] * W.E_CHARGE
        sp.append(W.Species(f"s{k}", q, W.M_E * (1 + 400 * k), 3e9 * (1 + k), src_vth=1e5))
    n = 8 * n_per
    tags = np.repeat(np.arange(8, dtype=np.uint8), n_per)
    vth = np.array([4e5 / np.sqrt(1 + 400 * k) for k in range(8)])[tags]
    w = W.make_custom(nc, dx, 0, 2e-12, sp, B=(0.3, 0.1, 0.2), capacity=n + 64, seed=88,
                      x=rng.random(n) * nc * dx, vx=vth * rng.standard_normal(n), vy=vth * rng.standard_normal(n),
                      vz=vth * rng.standard_normal(n), sp=tags)
    g, o = run_pair(w, 30)
    assert assert_state_equal(g, o, where="eight species")
    assert_moments = __import__("parity").assert_moments_close
    assert_moments(g, o, tol=1e-9)
    g.close()


def test_checkpoint_is_refused_while_the_field_is_frozen():
    """The blob holds no E (restart solves it from rho): under bit1_set_E(E, freeze) a restart would continue with the
    self-consistent field instead of the prescribed one, so bit1_checkpoint says BIT1_ERR_STATE until the field is
    released, and the context stays usable."""
    import torch
    from paper_2606_28534_b200.binding import Bit1, Bit1Error, ERR_STATE

    w = W.make_config(2, scale=1 / 64)
    g = Bit1(w)
    g.load()
    blob = torch.empty(g.checkpoint_size(), dtype=torch.uint8).pin_memory()
    E = np.linspace(-50.0, 50.0, w.nc + 1)
    g.set_E(E, freeze_field=True)
    g.step(3)
    with pytest.raises(Bit1Error) as e:
        g.checkpoint(blob)
    assert e.value.status == ERR_STATE
    assert np.array_equal(g.get_E(), E), "the refusal must not touch the prescribed field"
    g.step(2)                              # still running under the frozen field
    assert np.array_equal(g.get_E(), E)
    g.set_E(g.get_E(), freeze_field=False)  # released: the next step solves the field again
    g.step(1)
    g.checkpoint(blob)
    g.checkpoint_wait()
    g.step(4)
    g.sync()
    want = g.get_particles()
    h = Bit1(w)
    h.restart(blob)
    h.step(4)
    h.sync()
    got = h.get_particles()
    for k in want:
        assert np.array_equal(want[k], got[k]), k
    assert np.array_equal(g.get_E(), h.get_E())
    g.close()
    h.close()
