"""In-tree build of libgbfit.so (the C-ABI library of include/gbfit.h) with nvcc for sm_100a.

`python -m paper_2405_04690_b200.build` or `build()`; the .so lands beside this file so that it
travels with the source tree (it is git-ignored, not gpurun-ignored).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libgbfit.so")
SOURCES = ["gbfit.cu"]
HEADERS = ["gb_math.cuh", "gb_fast.cuh", "gb_sincos_poly.h", "gb_fft.cuh", "gb_band.cuh", "gb_temper.cuh", "gb_tables.hpp", os.path.join("..", "..", "include", "gbfit.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
    "--fmad=true",          # contraction is wanted everywhere except the carrier bin (explicit __dmul_rn there)
    "-Xptxas", "-v",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libgbfit.so cannot be built (there is no CPU fallback)")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu -> libgbfit.so.  Returns the library path."""
    if not force and not stale():
        return LIB
    cmd = [nvcc_path(), *NVCC_FLAGS, *[os.path.join(CSRC, s) for s in SOURCES], "-o", LIB + ".tmp"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libgbfit.so")
    os.replace(LIB + ".tmp", LIB)
    log = os.path.join(_HERE, "build_ptxas.log")
    with open(log, "w") as fh:
        fh.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose:
        sys.stderr.write(res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
