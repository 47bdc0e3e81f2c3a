"""Host-side logic of the command-line runner (python -m paper_2606_28534_b200): where the run comes back to the host,
and the crash-safe checkpoint file write.  No GPU."""
import os

import numpy as np

from paper_2606_28534_b200.__main__ import plan_stops, write_atomic


def test_stops_are_the_multiples_of_every_interval_and_the_last_step():
    assert plan_stops(0, 10) == [10]
    assert plan_stops(0, 1000, dmpstep=500) == [500, 1000]
    assert plan_stops(0, 1000, dmpstep=300, report=250) == [250, 300, 500, 600, 750, 900, 1000]
    assert plan_stops(500, 1000, dmpstep=500) == [1000]                 # restarted on a multiple: not repeated
    assert plan_stops(520, 1100, dmpstep=500, mvstep=200) == [600, 800, 1000, 1100]
    assert plan_stops(10, 10, dmpstep=5) == [] and plan_stops(10, 5) == []
    assert plan_stops(0, 7, dmpstep=0, report=0, mvstep=0) == [7]


def test_checkpoint_file_is_replaced_atomically(tmp_path):
    path = str(tmp_path / "bit1.ckpt")
    a = np.arange(1000, dtype=np.uint8)
    write_atomic(path, a)
    assert np.array_equal(np.fromfile(path, dtype=np.uint8), a)
    b = np.full(300, 7, dtype=np.uint8)
    write_atomic(path, b)                       # shorter file replaces the longer one completely
    assert np.array_equal(np.fromfile(path, dtype=np.uint8), b)
    assert not os.path.exists(path + ".part")


def test_a_failed_write_leaves_the_previous_checkpoint(tmp_path):
    path = str(tmp_path / "bit1.ckpt")
    write_atomic(path, np.arange(10, dtype=np.uint8))

    class Boom:
        def __buffer__(self, flags):
            raise RuntimeError("disk full")

    try:
        write_atomic(path, Boom())
    except Exception:
        pass
    assert np.array_equal(np.fromfile(path, dtype=np.uint8), np.arange(10, dtype=np.uint8))
