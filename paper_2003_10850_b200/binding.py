"""Thin ctypes binding of libsph.so (include/sph.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is no CPU fallback: if libsph.so is missing or no CUDA device is
present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsph.so")

COMPACT_NOALLOC_MAX = 1 << 26  # SPH_COMPACT_NOALLOC_MAX of include/sph.h
SPH_OK, SPH_E_ARG, SPH_E_CUDA, SPH_E_NOINDEX, SPH_E_OOM, SPH_E_INTERNAL, SPH_E_HRANGE, SPH_W_NOCONV = 0, 1, 2, 3, 4, 5, 6, 16
ST_CONVERGED, ST_BRACKET, ST_NOTCONV, ST_STALLED = 1 << 8, 1 << 9, 1 << 10, 1 << 11
KERNEL_CUBIC, KERNEL_WC6 = 0, 1

EXPORTS = ["sph_create", "sph_destroy", "sph_build_index", "sph_density", "sph_hydro_force", "sph_step_host",
           "sph_get_stats", "sph_velocity_gradients", "sph_hydro_force_improved", "sph_thermal_conduction",
           "sph_kdk_init", "sph_kdk_step", "sph_gravity_short", "sph_refresh_index", "sph_compact_flags", "sph_compact_flags_noalloc",
           "sph_last_error", "sph_version"]


class SphParams(C.Structure):
    _fields_ = [("kernel", C.c_int), ("box", C.c_float), ("gamma", C.c_float), ("alpha_visc", C.c_float),
                ("count_mode", C.c_int), ("max_iter", C.c_int), ("group_cap", C.c_int), ("group_node", C.c_int)]


class SphStats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("n", "n_nodes", "n_groups", "launches", "dens_evals", "dens_candidates",
                                         "dens_pairs", "force_candidates", "force_pairs")] + \
               [(k, C.c_float) for k in ("t_index_ms", "t_density_kernel_ms", "t_force_prep_ms", "t_force_kernel_ms")] + \
               [("node_pool_overflow", C.c_int64)]


class SphImprovedParams(C.Structure):
    _fields_ = [("alpha_min", C.c_float), ("alpha_max", C.c_float), ("decay_l", C.c_float), ("alpha_cond", C.c_float),
                ("balsara", C.c_int)]


class SphKdkParams(C.Structure):
    _fields_ = [("dt_max", C.c_float), ("n_bins", C.c_int), ("courant", C.c_float), ("eta", C.c_float),
                ("n_ngb_target", C.c_float), ("n_ngb_tol", C.c_float), ("refresh_max", C.c_int), ("rebuild_fraction", C.c_float),
                ("grav_G", C.c_float), ("grav_rs", C.c_float), ("grav_rcut", C.c_float), ("grav_eps", C.c_float), ("grav_theta", C.c_float)]


KDK_F32 = ("pos", "vel", "u", "h", "rho", "omega")
KDK_FIELDS = (("pos", 3), ("vel", 3), ("u", 1), ("h", 1), ("rho", 1), ("omega", 1), ("ngb", 1), ("acc", 3), ("dudt", 1), ("vsig", 1),
              ("vpred", 3), ("upred", 1), ("bin", 1), ("tbegin", 1), ("active", 1))


class SphKdkState(C.Structure):
    _fields_ = [(k, C.c_void_p) for k, _ in KDK_FIELDS]


class SphError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libsph status {code}: {msg}")
        self.code = code


_lib = None


def load():
    """Load libsph.so (built in-tree by paper_2003_10850_b200/build.py). Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not built: run `python -m paper_2003_10850_b200.build` "
                                    "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.sph_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(SphParams), C.c_void_p]
        lib.sph_destroy.argtypes = [C.c_void_p]
        lib.sph_build_index.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_float]
        lib.sph_density.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_float] + [C.c_void_p] * 5 + \
                                   [C.POINTER(C.c_int64)]
        lib.sph_hydro_force.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 8
        lib.sph_step_host.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p,
                                      C.c_int64, C.c_float, C.c_float] + [C.c_void_p] * 7 + [C.POINTER(C.c_int64)]
        lib.sph_get_stats.argtypes = [C.c_void_p, C.POINTER(SphStats)]
        lib.sph_last_error.argtypes = [C.c_void_p]
        lib.sph_last_error.restype = C.c_char_p
        lib.sph_version.restype = C.c_char_p
        lib.sph_velocity_gradients.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 5
        lib.sph_hydro_force_improved.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 8 + \
                                                [C.POINTER(SphImprovedParams)] + [C.c_void_p] * 4
        lib.sph_thermal_conduction.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 3 + [C.c_float, C.c_float, C.c_void_p]
        lib.sph_kdk_init.argtypes = [C.c_void_p, C.c_int64, C.c_float, C.POINTER(SphKdkParams), C.POINTER(SphKdkState)]
        lib.sph_kdk_step.argtypes = [C.c_void_p, C.c_int64, C.c_float, C.POINTER(SphKdkParams), C.POINTER(SphKdkState),
                                     C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        lib.sph_gravity_short.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_float] * 5 + [C.c_void_p]
        lib.sph_refresh_index.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
        for f in (lib.sph_compact_flags, lib.sph_compact_flags_noalloc):
            f.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        for name in EXPORTS[:16]:
            getattr(lib, name).restype = C.c_int
        _lib = lib
    return _lib


def _dev(t, dtype, name, numel=None):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def _host(t, dtype, name, numel):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous CPU tensor of dtype {dtype}")
    if t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


class Sph:
    """One libsph context (sph_create ... sph_destroy) bound to a torch CUDA stream."""

    def __init__(self, kernel=KERNEL_CUBIC, box=1.0, gamma=5.0 / 3.0, alpha_visc=1.0, count_mode=0, max_iter=64,
                 group_cap=0, group_node=0, stream: "torch.cuda.Stream | None" = None):
        self._lib = load()
        self._h = C.c_void_p()
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        p = SphParams(kernel, box, gamma, alpha_visc, count_mode, max_iter, group_cap, group_node)
        rc = self._lib.sph_create(C.byref(self._h), C.byref(p), C.c_void_p(self.stream.cuda_stream))
        if rc != SPH_OK:
            self._h = C.c_void_p()
            raise SphError(rc, "sph_create failed (no CUDA device? there is no CPU fallback)")
        self.n = 0

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.sph_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, allow=(SPH_OK,)):
        if rc not in allow:
            raise SphError(rc, self._lib.sph_last_error(self._h).decode())
        return rc

    # -- the three calls of the paper's statement of the problem -------------------------------
    def sph_build_index(self, pos, mass=None, mass_scalar=1.0):
        n = pos.shape[0]
        self._check(self._lib.sph_build_index(self._h, n, _dev(pos, torch.float32, "pos", 3 * n),
                                              _dev(mass, torch.float32, "mass", n), float(mass_scalar)))
        self.n = n

    def sph_refresh_index(self, pos):
        """Positions moved a little since sph_build_index: keep the tree, refresh the sorted positions, enlarge the cells."""
        n = pos.shape[0]
        self._check(self._lib.sph_refresh_index(self._h, n, _dev(pos, torch.float32, "pos", 3 * n)))

    def sph_compact_flags(self, flags, ids_out, count, noalloc=False):
        """ids_out[:count] = ascending indices of the non-zero flags (u32 0/1); count: u32 tensor of one element.
        noalloc=True: sph_compact_flags_noalloc (fixed device scratch, n <= COMPACT_NOALLOC_MAX, allocates nothing)."""
        n = flags.numel()
        fn = self._lib.sph_compact_flags_noalloc if noalloc else self._lib.sph_compact_flags
        self._check(fn(self._h, n, _dev(flags, torch.uint32, "flags", n), _dev(ids_out, torch.int32, "ids_out", n),
                       _dev(count, torch.uint32, "count", 1)))

    def sph_density(self, h, rho, omega, ngb_count, n_ngb_target, n_ngb_tol, active=None, status=None):
        """Returns the number of active particles that stopped without convergence."""
        n = self.n
        na = -1 if active is None else active.numel()
        unconv = C.c_int64(0)
        self._check(self._lib.sph_density(self._h, _dev(active, torch.int32, "active"), na, float(n_ngb_target),
                                          float(n_ngb_tol), _dev(h, torch.float32, "h", n),
                                          _dev(rho, torch.float32, "rho", n), _dev(omega, torch.float32, "omega", n),
                                          _dev(ngb_count, torch.int32, "ngb_count", n),
                                          _dev(status, torch.int32, "status", n), C.byref(unconv)),
                    allow=(SPH_OK, SPH_W_NOCONV))
        return int(unconv.value)

    def sph_hydro_force(self, vel, u, h, rho, omega, acc, dudt, vsig_max, active=None):
        n = self.n
        na = -1 if active is None else active.numel()
        self._check(self._lib.sph_hydro_force(self._h, _dev(active, torch.int32, "active"), na,
                                              _dev(vel, torch.float32, "vel", 3 * n), _dev(u, torch.float32, "u", n),
                                              _dev(h, torch.float32, "h", n), _dev(rho, torch.float32, "rho", n),
                                              _dev(omega, torch.float32, "omega", n),
                                              _dev(acc, torch.float32, "acc", 3 * n),
                                              _dev(dudt, torch.float32, "dudt", n),
                                              _dev(vsig_max, torch.float32, "vsig_max", n)))

    # -- improved-SPH extension (R17-R20) ----------------------------------------------
    def sph_velocity_gradients(self, vel, h, rho, divv, curlv, active=None):
        n = self.n
        na = -1 if active is None else active.numel()
        self._check(self._lib.sph_velocity_gradients(self._h, _dev(active, torch.int32, "active"), na,
                                                     _dev(vel, torch.float32, "vel", 3 * n), _dev(h, torch.float32, "h", n),
                                                     _dev(rho, torch.float32, "rho", n), _dev(divv, torch.float32, "divv", n),
                                                     _dev(curlv, torch.float32, "curlv", 3 * n)))

    def sph_hydro_force_improved(self, vel, u, h, rho, omega, alpha, divv, curlv, acc, dudt, vsig_max, dalpha_dt, active=None,
                                 alpha_min=0.02, alpha_max=3.0, decay_l=4.0, alpha_cond=0.25, balsara=True):
        n = self.n
        na = -1 if active is None else active.numel()
        ip = SphImprovedParams(alpha_min, alpha_max, decay_l, alpha_cond, int(bool(balsara)))
        f32 = torch.float32
        self._check(self._lib.sph_hydro_force_improved(
            self._h, _dev(active, torch.int32, "active"), na, _dev(vel, f32, "vel", 3 * n), _dev(u, f32, "u", n),
            _dev(h, f32, "h", n), _dev(rho, f32, "rho", n), _dev(omega, f32, "omega", n), _dev(alpha, f32, "alpha", n),
            _dev(divv, f32, "divv", n), _dev(curlv, f32, "curlv", 3 * n), C.byref(ip), _dev(acc, f32, "acc", 3 * n),
            _dev(dudt, f32, "dudt", n), _dev(vsig_max, f32, "vsig_max", n), _dev(dalpha_dt, f32, "dalpha_dt", n)))

    def sph_thermal_conduction(self, u, h, rho, dudt_cond, kappa0, kappa_exp=2.5, active=None):
        """R21: isotropic heat conduction as a further pair pass over the index."""
        n = self.n
        na = -1 if active is None else active.numel()
        f32 = torch.float32
        self._check(self._lib.sph_thermal_conduction(self._h, _dev(active, torch.int32, "active"), na, _dev(u, f32, "u", n),
                                                     _dev(h, f32, "h", n), _dev(rho, f32, "rho", n), float(kappa0), float(kappa_exp),
                                                     _dev(dudt_cond, f32, "dudt_cond", n)))

    def sph_gravity_short(self, acc_grav, G, r_s, r_cut, eps, theta, active=None):
        """R23: short-range Barnes-Hut gravity on the octree of the index (theta = 0: exact direct sum)."""
        n = self.n
        na = -1 if active is None else active.numel()
        self._check(self._lib.sph_gravity_short(self._h, _dev(active, torch.int32, "active"), na, float(G), float(r_s), float(r_cut),
                                                float(eps), float(theta), _dev(acc_grav, torch.float32, "acc_grav", 3 * n)))

    # -- kick-drift-kick driver with power-of-two time bins (R22) ---------------------------
    @staticmethod
    def _kdk_state(state: dict, n: int) -> "SphKdkState":
        st = SphKdkState()
        for k, w in KDK_FIELDS:
            dt = torch.int32 if k in ("ngb", "bin", "tbegin", "active") else torch.float32
            setattr(st, k, _dev(state[k], dt, k, w * n))
        return st

    def sph_kdk_init(self, state: dict, mass_scalar, dt_max, n_bins, n_ngb_target, n_ngb_tol, courant=0.3, eta=0.025,
                     refresh_max=16, rebuild_fraction=1.0 / 16, gravity=None):
        """gravity: None or dict(G, r_s, r_cut, eps, theta) -- short-range gravity added to the hydro acceleration."""
        n = state["pos"].shape[0]
        self._kdk_p = SphKdkParams(dt_max, n_bins, courant, eta, n_ngb_target, n_ngb_tol, refresh_max, rebuild_fraction,
                                   *([gravity[k] for k in ("G", "r_s", "r_cut", "eps", "theta")] if gravity else [0.0] * 5))
        st = self._kdk_state(state, n)
        self._check(self._lib.sph_kdk_init(self._h, n, float(mass_scalar), C.byref(self._kdk_p), C.byref(st)), allow=(SPH_OK, SPH_W_NOCONV))
        self.n = n

    def sph_kdk_step(self, state: dict, mass_scalar):
        """One step of the driver; returns (tick, n_active)."""
        n = state["pos"].shape[0]
        st = self._kdk_state(state, n)
        tick, na = C.c_int64(0), C.c_int64(0)
        self._check(self._lib.sph_kdk_step(self._h, n, float(mass_scalar), C.byref(self._kdk_p), C.byref(st), C.byref(tick), C.byref(na)),
                    allow=(SPH_OK, SPH_W_NOCONV))
        return int(tick.value), int(na.value)

    def sph_step_host(self, pos, vel, u, mass_scalar, h, rho, omega, ngb_count, acc, dudt, vsig, n_ngb_target,
                      n_ngb_tol, active=None):
        """Whole pass with HOST (ideally pinned) tensors; returns the unconverged count."""
        n = pos.shape[0]
        na = -1 if active is None else active.numel()
        unconv = C.c_int64(0)
        f32, i32 = torch.float32, torch.int32
        self._check(self._lib.sph_step_host(self._h, n, _host(pos, f32, "pos", 3 * n), _host(vel, f32, "vel", 3 * n),
                                            _host(u, f32, "u", n), float(mass_scalar),
                                            _host(active, i32, "active", na), na, float(n_ngb_target), float(n_ngb_tol),
                                            _host(h, f32, "h", n), _host(rho, f32, "rho", n),
                                            _host(omega, f32, "omega", n), _host(ngb_count, i32, "ngb_count", n),
                                            _host(acc, f32, "acc", 3 * n), _host(dudt, f32, "dudt", n),
                                            _host(vsig, f32, "vsig", n), C.byref(unconv)),
                    allow=(SPH_OK, SPH_W_NOCONV))
        self.n = n
        return int(unconv.value)

    def stats(self) -> dict:
        s = SphStats()
        self._check(self._lib.sph_get_stats(self._h, C.byref(s)))
        return {k: (int if t is C.c_int64 else float)(getattr(s, k)) for k, t in SphStats._fields_}


def version() -> str:
    return load().sph_version().decode()
