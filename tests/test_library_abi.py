"""-m "not gpu": libsph.so builds/loads and exports every symbol include/sph.h declares; host logic."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported():
    from paper_2003_10850_b200 import build

    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert {"sph_create", "sph_destroy", "sph_build_index", "sph_density", "sph_hydro_force", "sph_step_host",
            "sph_get_stats", "sph_fp32_peak", "sph_last_error", "sph_version"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    lib.sph_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.sph_version()


def test_binding_lists_the_same_entry_points():
    from paper_2003_10850_b200 import binding

    assert sorted(binding.EXPORTS) == _declared()


def test_no_cpu_fallback_without_device():
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2003_10850_b200 import binding

    lib = binding.load()
    h = ctypes.c_void_p()
    p = binding.SphParams(0, 1.0, 5.0 / 3.0, 1.0, 0, 64, 0)
    rc = lib.sph_create(ctypes.byref(h), ctypes.byref(p), None)
    assert rc == binding.SPH_E_CUDA and not h.value  # fails loudly, no fallback path
    assert lib.sph_create(None, ctypes.byref(p), None) == binding.SPH_E_ARG
    bad = binding.SphParams(5, 1.0, 5.0 / 3.0, 1.0, 0, 64, 0)
    assert lib.sph_create(ctypes.byref(h), ctypes.byref(bad), None) == binding.SPH_E_ARG


def test_product_does_not_import_oracle():
    """The CUDA path and the oracle share no code and neither imports the other."""
    pat = re.compile(r"(from|import)\s+oracle|sph_oracle|libsph_oracle|#include\s+\"[^\"]*oracle")
    pk = os.path.join(ROOT, "paper_2003_10850_b200")
    for dp, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dp, f)).read()), f
    assert not pat.search(open(os.path.join(ROOT, "include", "sph.h")).read())
    s = open(os.path.join(ROOT, "oracle", "sph_oracle.py")).read() + open(os.path.join(ROOT, "oracle", "sph_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2003_10850_b200", s, flags=re.M)
    assert "sph.h" not in s and "libsph.so" not in s and "csrc" not in s.replace("paper_2003_10850_b200/csrc", "")
