"""The C ABI from C: tests/c/abi_smoke.c includes include/sph.h, is compiled here with gcc against libsph.so and the
CUDA runtime, and drives create -> build_index -> density -> hydro_force -> get_stats plus the error paths without any
Python mirror of the structs in between."""
import os
import subprocess

import pytest

from paper_2003_10850_b200 import build

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_c_caller_runs_the_whole_path(tmp_path):
    lib = build.build()
    exe = str(tmp_path / "abi_smoke")
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    subprocess.check_call(["gcc", "-std=c99", "-O1", "-Wall", "-o", exe, os.path.join(ROOT, "tests", "c", "abi_smoke.c"),
                           "-I", os.path.join(ROOT, "include"), "-I", os.path.join(cuda, "include"), lib,
                           "-L", os.path.join(cuda, "lib64"), "-lcudart", "-lm",
                           "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.join(cuda, "lib64")])
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "abi_smoke ok" in r.stdout, r.stdout + r.stderr
