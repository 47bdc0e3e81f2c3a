"""Build libbit1.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

-fmad=false is mandatory: the arithmetic policy forbids FMA contraction so that the
particle state is bit-identical to the CPU oracle's.
"""
from __future__ import annotations

import hashlib
import os
import socket
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libbit1.so")
LIB_CHECKED = os.path.join(_HERE, "libbit1_checked.so")   # -DBIT1_CHECKED: index checks in the step kernels (common.cuh)
SOURCES = ["api.cu", "step_kernels.cu", "general_kernels.cu", "aux_kernels.cu", "field_static.cu"]
HEADERS = ["common.cuh", "device_math.cuh", "advance.cuh", "pipeline.cuh", "block_ops.cuh", "step_kernels.h", "aux_kernels.h",
           os.path.join("..", "..", "include", "bit1.h")]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-fmad=false", "-lineinfo",
              "-Xcompiler", "-fPIC,-ffp-contract=off", "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _fingerprint(checked: bool = False) -> str:
    """sha256 over everything the library is made from: sources, headers, flags, this file."""
    h = hashlib.sha256()
    for d in [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]:
        with open(d, "rb") as f:
            h.update(os.path.basename(d).encode() + b"\0" + f.read() + b"\0")
    h.update(" ".join(NVCC_FLAGS + (["-DBIT1_CHECKED"] if checked else [])).encode())
    return h.hexdigest()


def _stamp(lib: str):
    """(hostname, fingerprint) written next to the library by the build that made it, or (None, None)."""
    try:
        with open(lib + ".stamp") as f:
            host, fp = f.read().split()
        return host, fp
    except (OSError, ValueError):
        return None, None


def stale(lib: str = LIB) -> bool:
    """True unless `lib` exists and was built from exactly the present sources and flags (content hash, not mtimes: a
    tree that arrives with its library -- a gpurun snapshot, a fresh checkout next to an old build -- has arbitrary
    file times)."""
    if not os.path.exists(lib):
        return True
    return _stamp(lib)[1] != _fingerprint(checked=(lib == LIB_CHECKED))


def built_here(lib: str = LIB) -> bool:
    """The library was compiled on this host (its stamp says so)."""
    return os.path.exists(lib) and _stamp(lib)[0] == socket.gethostname()


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """checked=True builds libbit1_checked.so, the same sources with -DBIT1_CHECKED (profiles/r2_sanitizer.md)."""
    lib = LIB_CHECKED if checked else LIB
    if not force and not stale(lib):
        return lib
    objs = []
    log = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".checked.o" if checked else ".o"))
        cmd = [_nvcc(), *NVCC_FLAGS, *(["-DBIT1_CHECKED"] if checked else []), "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log.append(r.stderr)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib, *objs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    with open(os.path.join(CSRC, "ptxas_checked.log" if checked else "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    with open(lib + ".stamp", "w") as f:
        f.write(f"{socket.gethostname()} {_fingerprint(checked)}\n")
    if verbose:
        print("\n".join(log))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
