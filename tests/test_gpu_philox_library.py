"""Philox4x32-10 pinned to a library routine (SURVEY 8(c) "Pins"): cuRAND's device function curand_Philox4x32_10, compiled
into a small probe at test time, against the oracle's Philox on random counters and keys -- and, through the parity tests,
against the CUDA path's own."""
import ctypes as C
import os
import subprocess
import tempfile

import numpy as np
import pytest

from oracle import oracle as O

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_philox_equals_curand_device_function():
    nvcc = "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    with tempfile.TemporaryDirectory() as tmp:
        so = os.path.join(tmp, "libprobe.so")
        subprocess.run([nvcc, "-O2", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC",
                        os.path.join(HERE, "curand_philox_probe.cu"), "-o", so], check=True)
        lib = C.CDLL(so)
        n = 4096
        rng = np.random.default_rng(41)
        ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
        key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
        ctr[:4] = [[0, 0, 0, 0], [0xFFFFFFFF] * 4, [7, 3, 1, 0], [1, 0, 0, 0]]
        key[:4] = [[0, 0], [0xFFFFFFFF] * 2, [0x12345678, 0x9ABCDEF0], [0, 0]]
        out = np.zeros((n, 4), np.uint32)
        assert lib.curand_philox_probe(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, n) == 0
        for i in range(n):
            assert list(map(int, O.philox4x32_10(ctr[i], key[i]))) == out[i].tolist(), f"counter {ctr[i]}, key {key[i]}"
