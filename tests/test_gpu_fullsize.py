"""Parity at the size and launch configuration bench.py times (BASELINE.json configs[3]: 2e8 particles, 65536
cells, persistent grid of 2 CTAs per SM): properties that hold at any size, checked exactly, plus a random
sample of particles whose next step the CPU oracle computes one by one from the same state and field."""
import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _scale_for_this_box():
    """Full size or nothing: the test's name promises configs[3] at its full 2e8 particles, which needs about 30 GB of
    host memory for the input arrays and 30 GB of HBM for two copies of the state.  A smaller box skips, with the
    reason in the report, instead of quietly testing a quarter-size case under the full-size name."""
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 0
    import torch
    free, _ = torch.cuda.mem_get_info()
    if avail > 48e9 and free > 30e9:
        return 1.0
    reason = (f"full size needs > 48 GB of free host memory and > 30 GB of free HBM; this box has "
              f"{avail / 1e9:.0f} GB and {free / 1e9:.0f} GB")
    print("SKIPPED test_gpu_fullsize: " + reason)
    pytest.skip(reason)


def _check_invariants(w, p, rho, dens, m, n_expected, where):
    nc = w.nc
    n = p["x"].shape[0]
    assert n == n_expected, f"{where}: particle count {n} vs {n_expected}"
    cell = p["cell"]
    assert np.all(cell[1:] >= cell[:-1]), f"{where}: cells not sorted"
    inv_dx = 1.0 / w.dx
    c2 = np.minimum(np.maximum(p["x"] * inv_dx, 0.0), float(nc - 1)).astype(np.int32)
    assert np.array_equal(c2, cell), f"{where}: cell != floor(x/dx)"
    counts = np.bincount(cell, minlength=nc)
    assert np.array_equal(np.diff(p["cell_start"]), counts), f"{where}: cell_start vs histogram"
    assert p["cell_start"][0] == 0 and p["cell_start"][-1] == n
    # pids: unique
    seen = np.zeros(int(m["next_pid"]), np.uint8)
    seen[p["pid"]] += 1
    assert seen.max() == 1, f"{where}: duplicate pid"
    # exact charge conservation in fixed point: sum_j dens_s[j] = Q_s * N_s, rho = sum_s sign_s dens_s
    e, two40 = W.E_CHARGE, 1099511627776.0
    per = np.bincount(p["sp"], minlength=len(w.species))
    tot = 0
    for s, spc in enumerate(w.species):
        Q = int(np.rint((e * spc.weight) * two40))
        assert int(dens[s].sum()) == Q * int(per[s]), f"{where}: species {s} deposited charge"
        tot += int(np.sign(spc.q)) * Q * int(per[s])
    assert int(rho.sum()) == tot == m["rho_total"], f"{where}: total charge"
    sign = np.array([int(np.sign(s.q)) for s in w.species], np.int64)
    assert np.array_equal(rho, (sign[:, None] * dens).sum(axis=0)), f"{where}: rho != sum_s sign_s dens_s"


def test_config4_full_size_invariants_and_sampled_oracle_parity():
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    scale = _scale_for_this_box()
    w = W.make_config(4, scale=scale)
    g = Bit1(w)  # default variant and launch configuration: what bench.py runs
    g.load()
    n0 = w.n
    # (1) Step 1 from the seeded inputs alone (nothing taken from the CUDA path): the quiet start puts every ion on its
    # electron and neutrals carry no charge, so rho, phi and E are exactly zero at load; the oracle advances a sample of
    # the INPUT particles in that field and the GPU's first step must give the same bits for them.
    assert not g.get_rho().any() and not g.get_E().any(), "quiet start: the field at load is exactly zero"
    rng = np.random.default_rng(2606)
    idx0 = np.unique(rng.choice(n0, size=200_000, replace=False))
    ws = W.make_config(4, scale=scale, particles=False)
    ws.capacity = idx0.shape[0] + 4096
    o0 = Oracle(ws, load=False)
    o0.load(w.x[idx0], w.vx[idx0], w.vy[idx0], w.vz[idx0], w.sp[idx0], pid=idx0.astype(np.uint32))
    o0.set_E(np.zeros(w.nc + 1))
    o0.step(1, freeze_field=True)
    p0 = o0.particles()
    g.step(1)
    g.sync()
    first = g.get_particles(cell_start=False)
    where = np.full(int(g.get_moments()["next_pid"]), -1, np.int64)
    where[first["pid"]] = np.arange(first["pid"].shape[0])
    own = np.isin(p0["pid"], idx0)
    pos = where[p0["pid"][own]]
    assert np.all(pos >= 0) and int(own.sum()) == idx0.shape[0]
    for key in ("x", "vx", "vy", "vz", "cell", "sp"):
        assert np.array_equal(first[key][pos], p0[key][own]), f"step 1 from the inputs: {key} differs"
    assert np.all(np.diff(pos) > 0), "step 1 from the inputs: order differs from the oracle's stable sort"
    del first, where, o0, p0
    # (2) One step in a developed field: state and field of the GPU at step k are the oracle's inputs here
    k = 2
    g.step(k - 1)
    g.sync()
    m = g.get_moments()
    before = g.get_particles()
    E = g.get_E()
    # the field solve on 64 CTAs against the oracle's plain serial solve of the same rho (exact integers: any scan order
    # must give these bits)
    from oracle import oracle as OM
    ob = Oracle(W.make_config(4, scale=scale, particles=False), load=False)
    cst = ob.constants()
    phi_o, E_o = OM.poisson(w.nc, w.bc, cst["Kphi"], cst["KE"], g.get_rho())
    assert np.array_equal(E, E_o) and np.array_equal(g.get_phi(), phi_o), "field solve at full size"
    del ob
    _check_invariants(w, before, g.get_rho(), g.get_dens(), m, n0 + m["births"], f"step {k}")

    # a sample of the particles: random ones, plus the ones nearest to both walls (they are absorbed and
    # re-injected) -- the oracle advances exactly these from the same state in the same field
    rng = np.random.default_rng(20260628)
    idx = np.unique(np.concatenate([rng.choice(before["x"].shape[0], size=200_000, replace=False),
                                    np.arange(0, 20_000), np.arange(before["x"].shape[0] - 20_000,
                                                                    before["x"].shape[0])]))
    ws = W.make_config(4, scale=scale, particles=False)
    ws.capacity = idx.shape[0] + 4096
    o = Oracle(ws, load=False)
    o.load(before["x"][idx], before["vx"][idx], before["vy"][idx], before["vz"][idx], before["sp"][idx],
           pid=before["pid"][idx])
    o.set_E(E)
    o.set_step(k)
    o.step(1, freeze_field=True)
    po = o.particles()
    sample_pids = before["pid"][idx]
    del before

    g.step(1)
    g.sync()
    m = g.get_moments()
    after = g.get_particles()
    _check_invariants(w, after, g.get_rho(), g.get_dens(), m, n0 + m["births"], f"step {k + 1}")

    where = np.full(int(m["next_pid"]), -1, np.int64)
    where[after["pid"]] = np.arange(after["pid"].shape[0])
    parents = np.isin(po["pid"], sample_pids)   # the oracle's own births carry other pids
    pos = where[po["pid"][parents]]
    assert np.all(pos >= 0), "a sampled particle that survives in the oracle is missing on the GPU"
    assert int(parents.sum()) == idx.shape[0], "under SRC_SELF nobody dies"
    for key in ("x", "vx", "vy", "vz", "cell", "sp"):
        assert np.array_equal(after[key][pos], po[key][parents]), f"sampled particles: {key} differs"
    # the oracle lists them in its stable order; a sub-sequence of a stable sort is stably sorted the same way
    assert np.all(np.diff(pos) > 0), "sampled particles appear in another order than the oracle's stable sort"
    g.close()


def test_config4_full_size_every_element_after_three_steps():
    """The workload bench.py times, at full size, in its launch configuration: all 2e8 particles and every grid value
    compared with the oracle after 3 steps (about 40 GB of host memory, 16 s of oracle time; skipped on smaller boxes)."""
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1
    from parity import assert_state_equal

    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 0
    import torch
    free, _ = torch.cuda.mem_get_info()
    if avail < 80e9 or free < 30e9:
        pytest.skip("needs 80 GB of host memory and 30 GB of HBM")
    w = W.make_config(4)
    g = Bit1(w)
    g.load()
    g.step(3)
    g.sync()
    o = Oracle(w)
    o.step(3)
    exact = assert_state_equal(g, o, where="config 4 at full size, 3 steps, every element")
    assert exact, "fp64 state, phi and E are within tolerance but not bit-identical"
    g.close()
