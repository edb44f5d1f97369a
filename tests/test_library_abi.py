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
            "sph_get_stats", "sph_last_error", "sph_version"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    lib.sph_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.sph_version()


def test_binding_lists_the_same_entry_points():
    from paper_2003_10850_b200 import binding

    assert sorted(binding.EXPORTS) == _declared()


def test_struct_layout_matches_the_c_header(tmp_path):
    """The ctypes mirror of binding.py against the layout the C compiler gives include/sph.h (tests/c/abi_layout.c),
    field by field; the enums too.  The C caller itself runs in tests/test_gpu_abi_c.py."""
    import subprocess

    from paper_2003_10850_b200 import binding as B

    exe = str(tmp_path / "abi_layout")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-o", exe, os.path.join(ROOT, "tests", "c", "abi_layout.c"),
                           "-I", os.path.join(ROOT, "include")])
    out = dict(l.split(None, 1) for l in subprocess.check_output([exe], text=True).splitlines())
    for name, cls in (("sph_params", B.SphParams), ("sph_stats", B.SphStats), ("sph_improved_params", B.SphImprovedParams),
                      ("sph_kdk_params", B.SphKdkParams), ("sph_kdk_state", B.SphKdkState)):
        assert int(out[name]) == ctypes.sizeof(cls)
        fields = [f for f, _ in cls._fields_]
        assert sorted(k.split(".")[1] for k in out if k.startswith(name + ".")) == sorted(fields)
        for f in fields:
            assert int(out[f"{name}.{f}"]) == getattr(cls, f).offset, (name, f)
    assert [int(x) for x in out["status"].split()] == [B.SPH_OK, B.SPH_E_ARG, B.SPH_E_CUDA, B.SPH_E_NOINDEX, B.SPH_E_OOM,
                                                       B.SPH_E_INTERNAL, B.SPH_E_HRANGE, B.SPH_W_NOCONV]
    assert [int(x) for x in out["flags"].split()] == [B.ST_CONVERGED, B.ST_BRACKET, B.ST_NOTCONV, B.ST_STALLED]
    # the smoke caller compiles against the header, too (it runs on the GPU box)
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-c", "-o", str(tmp_path / "abi_smoke.o"),
                           os.path.join(ROOT, "tests", "c", "abi_smoke.c"), "-I", os.path.join(ROOT, "include"),
                           "-I", "/usr/local/cuda/include"])


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
