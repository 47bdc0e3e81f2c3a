"""Streaming checkpoints (SURVEY 8(f) NEXT-4, second half; PAPER.md:22, :41 SST; PAPER.md:57 record order;
PAPER.md:143-147 a consumer that reads checkpoints without interrupting the run): a consumer thread takes per-species
records in the paper's layout off a ring of pinned slots while bit1_step keeps running.  Every snapshot it sees is
complete and equals the synchronous bit1_export_species at that step, and that in turn equals the oracle's state."""
import hashlib
import threading
import time

import numpy as np
import pytest

from paper_2606_28534_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _digest(species_records):
    h = hashlib.sha256()
    for r in species_records:
        for k in ("counts", "x", "vx", "vy", "vz", "pid"):
            a = np.ascontiguousarray(r[k])
            if k == "counts":
                a = a.astype(np.int64)
            h.update(a.tobytes())
    return h.hexdigest()


@pytest.mark.parametrize("cfg,scale,kw", [(3, 1 / 64, dict(n0_scale=200.0, pair_source=True, recycle=True)),
                                           (5, 1 / 2048, dict(n0_scale=100.0))])
def test_consumer_thread_sees_complete_snapshots_equal_to_the_synchronous_export(cfg, scale, kw):
    import torch
    from oracle.oracle import Oracle
    from paper_2606_28534_b200.binding import Bit1, Bit1Error, ERR_STATE

    w = W.make_config(cfg, scale=scale, **kw)
    every, rounds = 4, 8
    ns = len(w.species)
    # reference: the same run, exported synchronously at the same steps (and checked against the oracle)
    ref = Bit1(w)
    ref.load()
    o = Oracle(w)
    want = {}
    for _ in range(rounds):
        ref.step(every)
        o.step(every)
        recs = [ref.export_species(s) for s in range(ns)]
        step = ref.get_moments()["step"]
        want[step] = _digest(recs)
        po = o.particles()
        for s in range(ns):
            sel = po["sp"] == s
            assert np.array_equal(recs[s]["x"], po["x"][sel]) and np.array_equal(recs[s]["pid"], po["pid"][sel])
            assert np.array_equal(recs[s]["counts"], np.bincount(po["cell"][sel], minlength=w.nc))
    ref.close()

    with pytest.raises(Bit1Error) as e:   # needs the device snapshot area
        g0 = Bit1(w)
        g0.stream_open(torch.empty(2 * 4096, dtype=torch.uint8).pin_memory(), 2)
    assert e.value.status == ERR_STATE
    g0.close()

    g = Bit1(w, checkpoint_staging=True)
    g.load()
    nslots = 3
    slot = (g.stream_slot_size() + 255) // 256 * 256
    ring = torch.empty(nslots * slot, dtype=torch.uint8).pin_memory()
    g.stream_open(ring, nslots)
    seen, stop, errors = {}, threading.Event(), []

    def consumer():
        last = 0
        try:
            while True:
                got = g.stream_acquire(last)
                if got is None:
                    if stop.is_set():
                        return
                    time.sleep(0.0005)
                    continue
                seq, snap = got
                assert seq > last
                time.sleep(0.003)   # a slow reader: the producer must stay off the held slot meanwhile
                for r in snap["species"]:
                    assert int(r["counts"].sum()) == r["x"].shape[0]
                    cells = np.minimum((r["x"] * (1.0 / w.dx)).astype(np.int64), w.nc - 1)
                    assert np.array_equal(np.bincount(cells, minlength=w.nc), r["counts"]) and np.all(np.diff(cells) >= 0)
                assert sum(r["x"].shape[0] for r in snap["species"]) == snap["n_total"]
                seen[snap["step"]] = _digest(snap["species"])
                last = seq
                g.stream_release(seq)
        except Exception as ex:   # surfaced by the main thread
            errors.append(ex)

    t = threading.Thread(target=consumer)
    t.start()
    for _ in range(rounds):
        g.step(every)
        g.stream_publish()     # returns with the copy in flight: the next round's steps overlap it
    g.checkpoint_wait()        # the last copy has landed and its sequence number is out
    stop.set()
    t.join()
    g.stream_close()
    g.close()
    assert not errors, errors[0]
    assert seen and every * rounds in seen, sorted(seen)   # the newest snapshot is never dropped
    for step, d in seen.items():
        assert d == want[step], f"snapshot of step {step} differs from the synchronous export"


def test_stream_digests_match_at_every_published_step():
    """Publish at the same steps as the synchronous reference and compare every snapshot the consumer got."""
    import torch
    from paper_2606_28534_b200.binding import Bit1

    w = W.make_config(3, scale=1 / 64, n0_scale=200.0, pair_source=True)
    every, rounds, ns = 5, 6, len(w.species)
    ref = Bit1(w)
    ref.load()
    want = {}
    for _ in range(rounds):
        ref.step(every)
        want[ref.get_moments()["step"]] = _digest([ref.export_species(s) for s in range(ns)])
    ref.close()
    g = Bit1(w, checkpoint_staging=True)
    g.load()
    slot = (g.stream_slot_size() + 255) // 256 * 256
    ring = torch.empty(2 * slot, dtype=torch.uint8).pin_memory()
    g.stream_open(ring, 2)
    seen, done = {}, threading.Event()

    def consumer():
        last = 0
        while True:
            got = g.stream_acquire(last)
            if got is None:
                if done.is_set():
                    return
                time.sleep(0.0002)
                continue
            last, snap = got
            seen[snap["step"]] = _digest(snap["species"])
            g.stream_release(last)

    t = threading.Thread(target=consumer)
    t.start()
    for _ in range(rounds):
        g.step(every)
        g.stream_publish()     # returns with the copy in flight; the next steps overlap it
    g.checkpoint_wait()        # the last copy has landed and its sequence number is out
    done.set()
    t.join()
    g.stream_close()
    g.close()
    assert len(seen) >= 1 and every * rounds in seen, sorted(seen)
    for step, d in seen.items():
        assert d == want[step], f"snapshot of step {step} differs from the synchronous export"
