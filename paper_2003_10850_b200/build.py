"""Build libsph.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsph.so")
SOURCES = ["sph_api.cu", "sph_index.cu", "sph_sort.cu", "sph_density.cu", "sph_force.cu", "sph_kdk.cu", "sph_gravity.cu"]
HEADERS = ["sph_internal.cuh", "sph_warp.cuh", os.path.join(ROOT, "include", "sph.h")]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Wno-deprecated-declarations", "-Xcompiler", "-Wno-deprecated-declarations",
           "--shared", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    for d in os.environ.get("SPH_DEFS", "").split():  # development: e.g. SPH_DEFS="-DSPH_CTAS=4 -DSPH_QCAP=48 -DSPH_LEAF=24 -DSPH_GBLOCK=2"
        cmd.insert(1, d)
    if os.environ.get("SPH_DEBUG"):  # device-side bounds asserts (development only)
        cmd.insert(1, "-DSPH_DEBUG=1")
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
