"""Shared comparison helpers for the GPU parity tests (CUDA path vs CPU oracle, same seeded inputs)."""
import numpy as np


def run_pair(w, nsteps, *, checkpoint_staging=False, chunk=None, **bit1_kw):
    """Run the CUDA path and the oracle side by side; returns (gpu, oracle)."""
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1

    g = Bit1(w, checkpoint_staging=checkpoint_staging, **bit1_kw)
    g.load()
    o = Oracle(w)
    if nsteps:
        g.step(nsteps)
        o.step(nsteps)
    g.sync(check_flags=False)
    return g, o


def assert_state_equal(g, o, *, tol_state=1e-12, where=""):
    """Bit-exact: counts, cell indices, sort order (pid/species sequence), cell_start, rho, dens, wall and
    event counters.  fp64 state within tol_state relative (readings A26/A27);
    returns True when the floats are bit-identical too."""
    w = o.w
    pg, po = g.get_particles(), o.particles()
    assert pg["x"].shape[0] == o.n, f"{where} particle count {pg['x'].shape[0]} vs {o.n}"
    for k in ("cell", "pid", "sp"):
        assert np.array_equal(pg[k], po[k]), f"{where} {k} differs (sort order / cell index)"
    assert np.array_equal(pg["cell_start"], o.cell_start()), f"{where} cell_start"
    assert np.array_equal(g.get_rho(), o.rho()), f"{where} rho"
    assert np.array_equal(g.get_dens(), o.dens()), f"{where} dens"
    L = w.nc * w.dx
    exact = True
    dx = np.abs(pg["x"] - po["x"])
    assert dx.max(initial=0.0) <= tol_state * L, f"{where} x off by {dx.max()}"
    exact &= bool(np.array_equal(pg["x"], po["x"]))
    vn = np.sqrt(po["vx"] ** 2 + po["vy"] ** 2 + po["vz"] ** 2)
    vth = np.array([max(s.src_vth, 1.0) for s in w.species])[po["sp"]]
    scale = np.maximum(vn, vth)
    for k in ("vx", "vy", "vz"):
        d = np.abs(pg[k] - po[k])
        assert np.all(d <= tol_state * scale), f"{where} {k} off by {d.max()}"
        exact &= bool(np.array_equal(pg[k], po[k]))
    eg, eo = g.get_E(), o.E()
    fg, fo = g.get_phi(), o.phi()
    assert np.allclose(eg, eo, rtol=0, atol=1e-12 * max(np.abs(eo).max(), 1e-300)), f"{where} E"
    assert np.allclose(fg, fo, rtol=0, atol=1e-12 * max(np.abs(fo).max(), 1e-300)), f"{where} phi"
    exact &= bool(np.array_equal(eg, eo) and np.array_equal(fg, fo))
    mg = g.get_moments()
    wc, wq = o.wall()
    d = o.diag()
    assert np.array_equal(mg["wall_count"], wc) and np.array_equal(mg["wall_charge"], wq), f"{where} wall"
    assert mg["next_pid"] == o.next_pid and mg["step"] == o.step_index, f"{where} next_pid/step"
    assert np.array_equal(mg["candidates"], d["candidates"]) and np.array_equal(mg["events"], d["events"]), \
        f"{where} MC event counters"
    assert (mg["births"], mg["reinject"], mg["nu_overflow"], mg["dir_fallback"], mg["escape"]) == \
        (d["births"], d["reinject"], d["nu_overflow"], d["dir_fallback"], d["escape"]), f"{where} diagnostics"
    assert mg["recycled"] == o.recycled, f"{where} recycling events"
    assert mg["flags"] == o.flagword, f"{where} flags {mg['flags']} vs {o.flagword}"
    assert mg["rho_total"] == int(o.rho().sum())
    return exact


def assert_moments_close(g, o, tol=1e-9):
    mg, mo = g.get_moments(density=True), o.moments()
    assert np.array_equal(mg["count"], mo["count"])
    for k in ("kinetic_J", "px"):
        ref = np.abs(mo["kinetic_J"]) if k == "kinetic_J" else np.abs(mo[k]) + 1e-30
        if k == "kinetic_J":
            assert np.all(np.abs(mg[k] - mo[k]) <= tol * ref), k
    # momentum: relative to m w N vth (its own value can cancel to ~0)
    w = o.w
    for s, spc in enumerate(w.species):
        scale = spc.m * spc.weight * max(int(mo["count"][s]), 1) * max(spc.src_vth, 1.0)
        assert abs(mg["px"][s] - mo["px"][s]) <= tol * scale
    assert abs(mg["field_J"] - mo["field_J"]) <= tol * max(abs(mo["field_J"]), 1e-300)
    for s in range(len(w.species)):
        ref = o.density(s)
        assert np.all(np.abs(mg["density"][s] - ref) <= tol * max(ref.max(), 1e-300))
