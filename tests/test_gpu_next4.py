"""export of the state in the paper's checkpoint layout (per species, the vector of
particle counts per cell, then the position and velocity records located by the offsets those counts give).  The
expected value is the definition written out: a filter of the oracle's particle arrays by species."""
import ctypes as C

import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W
from parity import run_pair

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,scale,kw,steps", [
    (2, 1 / 32, dict(pair_source=True, recycle=True), 40),    # deaths, births, a species that starts empty
    (3, 1 / 64, dict(n0_scale=200.0), 25),
    (4, 1 / 1024, dict(n0_scale=100.0), 10),                   # 195 k particles: many chunks, ragged tail
    (1, 1 / 16, {}, 5),
])
def test_export_equals_the_oracle_state_filtered_by_species(cfg, scale, kw, steps):
    w = W.make_config(cfg, scale=scale, **kw)
    if kw.get("recycle"):
        w.vx[w.sp == 1] *= 30.0
    g, o = run_pair(w, steps)
    po = o.particles()
    total = 0
    for s in range(len(w.species)):
        e = g.export_species(s)
        sel = po["sp"] == s
        assert e["x"].shape[0] == int(sel.sum())
        for k in ("x", "vx", "vy", "vz", "pid"):
            assert np.array_equal(e[k], po[k][sel]), f"species {s}: {k}"
        assert np.array_equal(e["counts"], np.bincount(po["cell"][sel], minlength=w.nc)), f"species {s}: counts"
        # the counts locate every cell's records: offsets = exclusive prefix sum
        off = np.concatenate([[0], np.cumsum(e["counts"])])
        cells = np.minimum((e["x"] * (1.0 / w.dx)).astype(np.int64), w.nc - 1)
        assert np.array_equal(np.repeat(np.arange(w.nc), e["counts"]), cells) and off[-1] == e["x"].shape[0]
        total += e["x"].shape[0]
    assert total == o.n
    # the export leaves the live state alone: the run goes on bit for bit
    g.step(3)
    o.step(3)
    from parity import assert_state_equal
    assert assert_state_equal(g, o, where="after export")
    g.close()


def test_export_reloaded_gives_the_same_charge_and_counts_and_argument_checks():
    from paper_2606_28534_b200 import binding as B

    w = W.make_config(3, scale=1 / 128, n0_scale=200.0)
    g, o = run_pair(w, 12)
    parts = [g.export_species(s) for s in range(len(w.species))]
    cat = lambda k: np.concatenate([p[k] for p in parts])
    sp = np.concatenate([np.full(p["x"].shape[0], s, np.uint8) for s, p in enumerate(parts)])
    h = B.Bit1(w)
    h.load_particles(cat("x"), cat("vx"), cat("vy"), cat("vz"), sp, pid=cat("pid"))
    assert np.array_equal(h.get_rho(), g.get_rho()) and np.array_equal(h.get_dens(), g.get_dens())
    assert np.array_equal(h.get_count()[2], g.get_count()[2])
    assert np.array_equal(np.sort(h.get_particles()["pid"]), np.sort(g.get_particles()["pid"]))
    h.close()
    n = C.c_uint64()
    L = g.lib
    assert L.bit1_export_species(g.h, 9, 0, C.byref(n), None, None, None, None, None, None) == B.ERR_INVALID_ARG
    assert L.bit1_export_species(g.h, 0, 0, None, None, None, None, None, None, None) == B.ERR_INVALID_ARG
    x = np.zeros(4)
    assert L.bit1_export_species(g.h, 0, 4, C.byref(n), None, x.ctypes.data, None, None, None, None) == B.ERR_CAPACITY
    assert n.value == parts[0]["x"].shape[0]
    g.close()
