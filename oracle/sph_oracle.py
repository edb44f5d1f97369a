"""ctypes wrapper of oracle/sph_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2003_10850_b200 (the CUDA path) and the
CUDA path imports nothing from here.  See the header of sph_oracle.c for authority and pins.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sph_oracle.c")
_LIB = os.path.join(_HERE, "libsph_oracle.so")

F_CONVERGED, F_BRACKET, F_NOTCONV, F_STALLED = 1, 2, 4, 8
E_RADIUS, E_BAND, E_BRANCH = 1, 2, 4


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp (no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


class _Params(C.Structure):
    _fields_ = [("kernel", C.c_int), ("box", C.c_double), ("gamma", C.c_double), ("alpha", C.c_double),
                ("count_mode", C.c_int), ("max_iter", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        for name in ("orc_kernel_w", "orc_kernel_dw"):
            getattr(_lib, name).restype = C.c_double
            getattr(_lib, name).argtypes = [C.c_int, C.c_double]
        _lib.orc_kernel_sigma.restype = C.c_double
        _lib.orc_kernel_sigma.argtypes = [C.c_int]
        for name in ("orc_W", "orc_dWdr", "orc_dWdH"):
            getattr(_lib, name).restype = C.c_double
            getattr(_lib, name).argtypes = [C.c_int, C.c_double, C.c_double]
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a, dtype):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data_as(C.c_void_p)


def _params(kernel, box, gamma, alpha, count_mode, max_iter):
    return _Params(int(kernel), float(box), float(gamma), float(alpha), int(count_mode), int(max_iter))


def kernel_w(k, q):
    return lib().orc_kernel_w(int(k), float(q))


def kernel_dw(k, q):
    return lib().orc_kernel_dw(int(k), float(q))


def kernel_sigma(k):
    return lib().orc_kernel_sigma(int(k))


def W(k, r, H):
    return lib().orc_W(int(k), float(r), float(H))


def dWdr(k, r, H):
    return lib().orc_dWdr(int(k), float(r), float(H))


def dWdH(k, r, H):
    return lib().orc_dWdH(int(k), float(r), float(H))


def density_eval(pos, h, *, kernel, box=1.0, mass=None, mass_scalar=1.0, active=None, brute=False,
                 cell_hint=None):
    """One evaluation at the given fp32 support radii. Returns dict of fp64 arrays (per active)."""
    pos_, ppos = _p(pos, np.float32)
    h_, ph = _p(h, np.float32)
    m_, pm = _p(mass, np.float32)
    act_, pact = _p(active, np.int32)
    n = pos_.shape[0]
    na = n if act_ is None else act_.shape[0]
    out = {k: np.zeros(na, np.float64) for k in ("S", "Dp", "rho", "drho", "Nw")}
    out["Nint"] = np.zeros(na, np.int32)
    out["edge"] = np.zeros(na, np.uint8)
    prm = _params(kernel, box, 5.0 / 3.0, 1.0, 0, 64)
    if cell_hint is None:
        cell_hint = float(np.median(h_)) if n else box
    lib().orc_density_eval(C.byref(prm), C.c_int64(n), ppos, pm, C.c_double(mass_scalar), ph, pact,
                           C.c_int64(na), C.c_int(int(brute)), C.c_double(cell_hint),
                           *[out[k].ctypes.data_as(C.c_void_p) for k in ("S", "Dp", "rho", "drho", "Nw", "Nint", "edge")])
    H = h_.astype(np.float64) if act_ is None else h_.astype(np.float64)[act_]
    out["H"] = H
    out["omega"] = 1.0 + H / (3.0 * out["rho"]) * out["drho"]  # grad-h factor (R1), as in orc_density
    return out


def density(pos, h_guess, *, kernel, n_target, n_tol, box=1.0, mass=None, mass_scalar=1.0, active=None,
            count_mode=0, max_iter=64, brute=False, cell_hint=None):
    """The h iteration + density. Returns dict: H, rho, omega, Nw (fp64), Nint, iters, flags (int32), edge (uint8), n_evals."""
    pos_, ppos = _p(pos, np.float32)
    h_, ph = _p(h_guess, np.float32)
    m_, pm = _p(mass, np.float32)
    act_, pact = _p(active, np.int32)
    n = pos_.shape[0]
    na = n if act_ is None else act_.shape[0]
    out = {k: np.zeros(na, np.float64) for k in ("H", "rho", "omega", "Nw")}
    for k in ("Nint", "iters", "flags"):
        out[k] = np.zeros(na, np.int32)
    out["edge"] = np.zeros(na, np.uint8)
    nev = C.c_int64(0)
    prm = _params(kernel, box, 5.0 / 3.0, 1.0, count_mode, max_iter)
    if cell_hint is None:
        cell_hint = float(np.median(h_)) if n else box
    lib().orc_density(C.byref(prm), C.c_int64(n), ppos, pm, C.c_double(mass_scalar), ph, pact, C.c_int64(na),
                      C.c_double(n_target), C.c_double(n_tol), C.c_int(int(brute)), C.c_double(cell_hint),
                      *[out[k].ctypes.data_as(C.c_void_p) for k in ("H", "rho", "omega", "Nw", "Nint", "iters", "flags", "edge")],
                      C.byref(nev))
    out["n_evals"] = int(nev.value)
    return out


def hydro_force(pos, vel, u, h, rho, omega, *, kernel, box=1.0, gamma=5.0 / 3.0, alpha=1.0, mass=None,
                mass_scalar=1.0, active=None, brute=False, cell_hint=None):
    """Symmetric hydro-force pair sum. Returns dict: acc (na,3), dudt, vsig, asum, dusum, duvisc, asq, dusq (fp64),
    npair (int64), edge.  asum/dusum are the sums of |pair term|, asq/dusq of (pair term)^2 (tolerances, R15)."""
    pos_, ppos = _p(pos, np.float32)
    vel_, pvel = _p(vel, np.float32)
    u_, pu = _p(u, np.float32)
    h_, ph = _p(h, np.float32)
    rho_, prho = _p(rho, np.float32)
    om_, pom = _p(omega, np.float32)
    m_, pm = _p(mass, np.float32)
    act_, pact = _p(active, np.int32)
    n = pos_.shape[0]
    na = n if act_ is None else act_.shape[0]
    out = {"acc": np.zeros((na, 3), np.float64)}
    for k in ("dudt", "vsig", "asum", "dusum", "duvisc", "asq", "dusq"):
        out[k] = np.zeros(na, np.float64)
    out["npair"] = np.zeros(na, np.int64)
    out["edge"] = np.zeros(na, np.uint8)
    prm = _params(kernel, box, gamma, alpha, 0, 64)
    if cell_hint is None:
        cell_hint = float(np.median(h_)) if n else box
    lib().orc_hydro_force(C.byref(prm), C.c_int64(n), ppos, pvel, pu, pm, C.c_double(mass_scalar), ph, prho, pom,
                          pact, C.c_int64(na), C.c_int(int(brute)), C.c_double(cell_hint),
                          *[out[k].ctypes.data_as(C.c_void_p) for k in ("acc", "dudt", "vsig", "asum", "dusum", "duvisc", "npair", "edge", "asq", "dusq")])
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))


# ---------------------------------------------------------------- improved-SPH extension (R17-R20)
class _Improved(C.Structure):
    _fields_ = [("alpha_min", C.c_double), ("alpha_max", C.c_double), ("decay_l", C.c_double), ("alpha_cond", C.c_double),
                ("balsara", C.c_int)]


def velocity_gradients(pos, vel, h, rho, *, kernel, box=1.0, mass=None, mass_scalar=1.0, active=None):
    """R17: div v and curl v with the particle's own support radius (brute force over all j). Returns dict divv (na), curlv (na,3)."""
    pos_, ppos = _p(pos, np.float32)
    vel_, pvel = _p(vel, np.float32)
    h_, ph = _p(h, np.float32)
    rho_, prho = _p(rho, np.float32)
    m_, pm = _p(mass, np.float32)
    act_, pact = _p(active, np.int32)
    n = pos_.shape[0]
    na = n if act_ is None else act_.shape[0]
    out = {"divv": np.zeros(na, np.float64), "curlv": np.zeros((na, 3), np.float64)}
    prm = _params(kernel, box, 5.0 / 3.0, 1.0, 0, 64)
    lib().orc_velocity_gradients(C.byref(prm), C.c_int64(n), ppos, pvel, pm, C.c_double(mass_scalar), ph, prho, pact,
                                 C.c_int64(na), out["divv"].ctypes.data_as(C.c_void_p), out["curlv"].ctypes.data_as(C.c_void_p))
    return out


def hydro_force_improved(pos, vel, u, h, rho, omega, alpha, divv, curlv, *, kernel, box=1.0, gamma=5.0 / 3.0, mass=None,
                         mass_scalar=1.0, active=None, alpha_min=0.02, alpha_max=3.0, decay_l=4.0, alpha_cond=0.25, balsara=True):
    """R8-R12 with R18-R20 (brute force over all j). Returns dict acc (na,3), dudt, vsig, dalpha, asum, dusum, asq, dusq, ducond."""
    arrs = [_p(a, np.float32) for a in (pos, vel, u, h, rho, omega, alpha, divv, curlv)]
    m_, pm = _p(mass, np.float32)
    act_, pact = _p(active, np.int32)
    n = arrs[0][0].shape[0]
    na = n if act_ is None else act_.shape[0]
    out = {"acc": np.zeros((na, 3), np.float64)}
    for k in ("dudt", "vsig", "dalpha", "asum", "dusum", "asq", "dusq", "ducond"):
        out[k] = np.zeros(na, np.float64)
    prm = _params(kernel, box, gamma, 1.0, 0, 64)
    q = _Improved(alpha_min, alpha_max, decay_l, alpha_cond, int(bool(balsara)))
    (_, ppos), (_, pvel), (_, pu), (_, ph), (_, prho), (_, pom), (_, pal), (_, pdv), (_, pcv) = arrs
    lib().orc_hydro_force_improved(C.byref(prm), C.byref(q), C.c_int64(n), ppos, pvel, pu, pm, C.c_double(mass_scalar), ph, prho,
                                   pom, pal, pdv, pcv, pact, C.c_int64(na),
                                   *[out[k].ctypes.data_as(C.c_void_p) for k in ("acc", "dudt", "vsig", "dalpha", "asum", "dusum", "asq", "dusq", "ducond")])
    return out


def thermal_conduction(pos, u, h, rho, *, kernel, kappa0, kappa_exp=2.5, box=1.0, mass=None, mass_scalar=1.0, active=None):
    """R21: isotropic heat conduction pair sum (brute force over all j). Returns dict dudt, dusum, dusq (fp64, per active)."""
    pos_, ppos = _p(pos, np.float32)
    u_, pu = _p(u, np.float32)
    h_, ph = _p(h, np.float32)
    rho_, prho = _p(rho, np.float32)
    m_, pm = _p(mass, np.float32)
    act_, pact = _p(active, np.int32)
    n = pos_.shape[0]
    na = n if act_ is None else act_.shape[0]
    out = {k: np.zeros(na, np.float64) for k in ("dudt", "dusum", "dusq")}
    prm = _params(kernel, box, 5.0 / 3.0, 1.0, 0, 64)
    lib().orc_thermal_conduction(C.byref(prm), C.c_int64(n), ppos, pu, pm, C.c_double(mass_scalar), ph, prho,
                                 C.c_double(kappa0), C.c_double(kappa_exp), pact, C.c_int64(na),
                                 *[out[k].ctypes.data_as(C.c_void_p) for k in ("dudt", "dusum", "dusq")])
    return out


def gravity_short(pos, *, G, r_s, r_cut, eps, box=1.0, mass=None, mass_scalar=1.0, active=None):
    """R23: short-range (TreePM) gravity by direct summation. Returns dict acc (na,3), asum (sum of |pair terms|)."""
    pos_, ppos = _p(pos, np.float32)
    m_, pm = _p(mass, np.float32)
    act_, pact = _p(active, np.int32)
    n = pos_.shape[0]
    na = n if act_ is None else act_.shape[0]
    out = {"acc": np.zeros((na, 3), np.float64), "asum": np.zeros(na, np.float64)}
    prm = _params(0, box, 5.0 / 3.0, 1.0, 0, 64)
    lib().orc_gravity_short(C.byref(prm), C.c_int64(n), ppos, pm, C.c_double(mass_scalar), C.c_double(G), C.c_double(r_s),
                            C.c_double(r_cut), C.c_double(eps), pact, C.c_int64(na), out["acc"].ctypes.data_as(C.c_void_p),
                            out["asum"].ctypes.data_as(C.c_void_p))
    return out
