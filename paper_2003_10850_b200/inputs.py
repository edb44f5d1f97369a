"""Seeded synthetic particle sets (inputs only: no SPH arithmetic lives here).

The paper measures on Magneticum snapshots (PAPER.md:47 §1, :118 §3.1, :138 §3.2) that are
not available; these generators take their *shape* (near-homogeneous initial conditions,
late-time haloes + background, time-bin selected active cores: PAPER.md:31 Fig. 1, :37 §1,
:84-86 §2.2) and stand in for them.  The recipe is stated in DESIGN.md "Input recipe" and is
the five configs of BASELINE.json.  Both the oracle (tests, bench cpu_baseline) and the CUDA
path consume the fp32 arrays produced here; the inputs are *defined* as those fp32 arrays.

Every generator takes the particle count so that the tests can run scaled-down sets that
the fp64 oracle finishes in seconds.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SEED_BASE = 200310850  # arxiv id 2003.10850; seed = SEED_BASE + config number

KERNEL_CUBIC = 0
KERNEL_WC6 = 1


@dataclasses.dataclass
class ParticleSet:
    """fp32 inputs of one config (box L = 1, equal masses m = 1/N)."""

    name: str
    pos: np.ndarray  # (N,3) float32 in [0,1)
    vel: np.ndarray  # (N,3) float32
    u: np.ndarray  # (N,) float32 specific internal energy
    h_guess: np.ndarray  # (N,) float32 support-radius guess handed to both sides
    mass: float  # scalar particle mass (1/N)
    kernel: int  # KERNEL_CUBIC / KERNEL_WC6
    n_ngb: float  # neighbour-number target N_t
    n_tol: float  # tolerance on the neighbour number
    box: float = 1.0
    active: np.ndarray | None = None  # int32 ids, None = all active
    aux: dict = dataclasses.field(default_factory=dict)  # generator-side metadata (halo ids ...)

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])


def h_of_number_density(n_density, n_ngb):
    """Support radius whose sphere holds n_ngb particles at number density n_density (guess recipe)."""
    return (3.0 * n_ngb / (4.0 * math.pi * n_density)) ** (1.0 / 3.0)


def _wrap01(x: np.ndarray) -> np.ndarray:
    """Wrap to [0,1) and make sure the fp32 cast cannot round up to 1.0."""
    x = x - np.floor(x)
    x32 = x.astype(np.float32)
    x32[x32 >= np.float32(1.0)] = np.float32(0.0)
    return x32


def _jittered_lattice(rng, n_side: int) -> np.ndarray:
    d = 1.0 / n_side
    g = (np.arange(n_side) + 0.5) * d
    zz, yy, xx = np.meshgrid(g, g, g, indexing="ij")
    p = np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1)
    p = p + rng.uniform(-0.25, 0.25, size=p.shape) * d
    return _wrap01(p)


def _isotropic(rng, n: int) -> np.ndarray:
    ct = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * math.pi, n)
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    return np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)


def _loguniform(rng, lo, hi, n):
    return np.exp(rng.uniform(math.log(lo), math.log(hi), n))


def config1(n_side: int = 16, seed: int | None = None) -> ParticleSet:
    """C1: n_side^3 jittered lattice, u=1, v=0, cubic spline, N_t = 64 +- 2 (BASELINE.json configs[0])."""
    rng = np.random.default_rng(SEED_BASE + 1 if seed is None else seed)
    pos = _jittered_lattice(rng, n_side)
    n = pos.shape[0]
    h0 = h_of_number_density(float(n), 64.0)
    hg = (h0 * np.exp(rng.uniform(-0.1, 0.1, n))).astype(np.float32)
    return ParticleSet("C1", pos, np.zeros((n, 3), np.float32), np.ones(n, np.float32), hg,
                       1.0 / n, KERNEL_CUBIC, 64.0, 2.0)


def config2(n_side: int = 64, seed: int | None = None) -> ParticleSet:
    """C2: n_side^3 jittered lattice, v~N(0,0.1), u log-uniform [0.5,2], cubic, 64 +- 2 (configs[1])."""
    rng = np.random.default_rng(SEED_BASE + 2 if seed is None else seed)
    pos = _jittered_lattice(rng, n_side)
    n = pos.shape[0]
    vel = rng.normal(0.0, 0.1, (n, 3)).astype(np.float32)
    u = _loguniform(rng, 0.5, 2.0, n).astype(np.float32)
    h0 = h_of_number_density(float(n), 64.0)
    hg = (h0 * np.exp(rng.uniform(-0.1, 0.1, n))).astype(np.float32)
    return ParticleSet("C2", pos, vel, u, hg, 1.0 / n, KERNEL_CUBIC, 64.0, 2.0)


def _analytic_density_guess(pos64, n_bg, centres, r_cut, profile, n_ngb, rng, spread=0.1):
    """h guess from the generator's analytic number-density field: background + every
    clump whose cut radius reaches the particle (profile(k, r) = number density of clump k)."""
    from scipy.spatial import cKDTree

    n = pos64.shape[0]
    dens = np.full(n, float(n_bg))
    if len(centres):
        tree_p = cKDTree(pos64, boxsize=1.0)
        order = np.argsort(-r_cut)
        for k in order:
            idx = tree_p.query_ball_point(centres[k] % 1.0, r_cut[k])
            if not idx:
                continue
            idx = np.asarray(idx)
            d = pos64[idx] - centres[k]
            d -= np.round(d)
            r = np.sqrt((d * d).sum(1))
            dens[idx] += profile(k, r)
    h = h_of_number_density(dens, n_ngb) * np.exp(rng.uniform(-spread, spread, n))
    return np.minimum(h, 0.45).astype(np.float32), dens


def config3(n: int = 1 << 21, n_spheres: int = 200, seed: int | None = None) -> ParticleSet:
    """C3: half uniform, half in Plummer spheres (a log-uniform [0.005,0.02]); cubic, 64 +- 2 (configs[2])."""
    rng = np.random.default_rng(SEED_BASE + 3 if seed is None else seed)
    n_bg = n // 2
    n_cl = n - n_bg
    per = np.full(n_spheres, n_cl // n_spheres)
    per[: n_cl - per.sum()] += 1
    a = _loguniform(rng, 0.005, 0.02, n_spheres)
    centres = rng.uniform(0.0, 1.0, (n_spheres, 3))
    parts = [rng.uniform(0.0, 1.0, (n_bg, 3))]
    for k in range(n_spheres):
        x = rng.uniform(1e-12, 1.0, per[k])
        r = a[k] / np.sqrt(x ** (-2.0 / 3.0) - 1.0)
        parts.append(centres[k] + r[:, None] * _isotropic(rng, per[k]))
    pos64 = np.concatenate(parts) % 1.0
    pos = _wrap01(pos64)
    vel = rng.normal(0.0, 0.3, (n, 3)).astype(np.float32)
    u = _loguniform(rng, 0.5, 2.0, n).astype(np.float32)

    def profile(k, r):
        return 3.0 * per[k] / (4.0 * math.pi * a[k] ** 3) * (1.0 + (r / a[k]) ** 2) ** -2.5

    hg, nd = _analytic_density_guess(pos.astype(np.float64), n_bg, centres, 30.0 * a, profile, 64.0, rng)
    halo = np.concatenate([np.full(n_bg, -1), np.repeat(np.arange(n_spheres), per)]).astype(np.int32)
    return ParticleSet("C3", pos, vel, u, hg, 1.0 / n, KERNEL_CUBIC, 64.0, 2.0,
                       aux={"halo": halo, "a": a, "centres": centres, "per": per, "n_density": nd})


def _nfw_m(x):
    return np.log1p(x) - x / (1.0 + x)


def _nfw_invert(y):
    """x with ln(1+x) - x/(1+x) = y (vectorised bisection + Newton polish, generator side only)."""
    lo = np.zeros_like(y)
    hi = np.full_like(y, 64.0)
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        big = _nfw_m(mid) > y
        hi = np.where(big, mid, hi)
        lo = np.where(big, lo, mid)
    return 0.5 * (lo + hi)


def config4(n: int = 10_000_000, n_halos: int = 2000, seed: int | None = None,
            m_lo: float = 320.0, m_hi: float = 1.0e6) -> ParticleSet:
    """C4: 30% uniform background + 70% in NFW haloes (c~U(5,15), dN/dM ~ M^-1.9); Wendland C6, 295 +- 2 (configs[3])."""
    rng = np.random.default_rng(SEED_BASE + 4 if seed is None else seed)
    n_bg = int(round(0.3 * n))
    n_cl = n - n_bg
    # power-law particle numbers, slope -1.9 on [m_lo, m_hi], rescaled to sum n_cl
    s = -1.9 + 1.0
    uu = rng.uniform(0.0, 1.0, n_halos)
    mm = (m_lo ** s + uu * (m_hi ** s - m_lo ** s)) ** (1.0 / s)
    mm *= n_cl / mm.sum()
    per = np.floor(mm).astype(np.int64)
    rest = n_cl - per.sum()
    per[np.argsort(-(mm - per))[:rest]] += 1
    conc = rng.uniform(5.0, 15.0, n_halos)
    # M = (4 pi / 3) 200 rho_mean r_vir^3 with rho_mean = 1, M = per / n
    r_vir = (3.0 * (per / float(n)) / (800.0 * math.pi)) ** (1.0 / 3.0)
    r_s = r_vir / conc
    centres = rng.uniform(0.0, 1.0, (n_halos, 3))
    parts = [rng.uniform(0.0, 1.0, (n_bg, 3))]
    radii = [np.zeros(n_bg)]
    for k in range(n_halos):
        y = rng.uniform(0.0, 1.0, per[k]) * _nfw_m(conc[k])
        r = r_s[k] * _nfw_invert(y)
        radii.append(r)
        parts.append(centres[k] + r[:, None] * _isotropic(rng, per[k]))
    pos = _wrap01(np.concatenate(parts))
    vel = rng.normal(0.0, 0.3, (n, 3)).astype(np.float32)
    u = _loguniform(rng, 0.5, 2.0, n).astype(np.float32)
    mc = _nfw_m(conc)

    def profile(k, r):
        x = np.maximum(r / r_s[k], 1e-4)
        return per[k] / (4.0 * math.pi * r_s[k] ** 3 * mc[k]) / (x * (1.0 + x) ** 2)

    hg, nd = _analytic_density_guess(pos.astype(np.float64), n_bg, centres, r_vir, profile, 295.0, rng)
    halo = np.concatenate([np.full(n_bg, -1), np.repeat(np.arange(n_halos), per)]).astype(np.int32)
    return ParticleSet("C4", pos, vel, u, hg, 1.0 / n, KERNEL_WC6, 295.0, 2.0,
                       aux={"halo": halo, "radius": np.concatenate(radii), "per": per, "conc": conc,
                            "r_s": r_s, "r_vir": r_vir, "centres": centres, "n_bg": n_bg, "n_density": nd})


def select_active_by_timebin(ps: ParticleSet, n_active: int) -> np.ndarray:
    """C5 active list: t_i ~ 1/sqrt(mean halo density inside r_i) from the generator's analytic NFW
    profile, power-of-two bins (PAPER.md:37 §1, :84-86 §2.2); lowest bins first, the last bin
    cut by particle id to exactly n_active ids.  Returned sorted by particle id (int32)."""
    aux = ps.aux
    halo = aux["halo"]
    n = ps.n
    rho_in = np.full(n, aux["n_bg"] / float(n))
    inh = halo >= 0
    k = halo[inh]
    x = np.maximum(aux["radius"][inh] / aux["r_s"][k], 1e-4)
    m_in = aux["per"][k] / float(n) * _nfw_m(x) / _nfw_m(aux["conc"][k])
    rho_in[inh] += m_in / (4.0 / 3.0 * math.pi * (x * aux["r_s"][k]) ** 3)
    t = 1.0 / np.sqrt(rho_in)
    b = np.floor(np.log2(t / t.min())).astype(np.int64)
    order = np.lexsort((np.arange(n), b))  # by bin, then by id
    return np.sort(order[:n_active]).astype(np.int32)


def config5_active(ps4: ParticleSet, frac: float = 0.01) -> np.ndarray:
    """C5 (configs[4]): 1% of the C4 set active, chosen by time-step bin of the halo cores."""
    return select_active_by_timebin(ps4, int(round(frac * ps4.n)))


def perturb_h(h: np.ndarray, ids: np.ndarray, seed: int, spread: float = 0.05) -> np.ndarray:
    """C5 guess for the active particles: converged H * exp(U(-spread, spread))."""
    rng = np.random.default_rng(seed)
    out = h.copy()
    out[ids] = (h[ids].astype(np.float64) * np.exp(rng.uniform(-spread, spread, len(ids)))).astype(np.float32)
    return out


def two_particles(r: float, h1: float, h2: float, u1=1.0, u2=1.0, v1=(0, 0, 0), v2=(0, 0, 0)):
    """Tiny hand-computable set used by the oracle pins."""
    pos = np.array([[0.25, 0.5, 0.5], [0.25 + r, 0.5, 0.5]], np.float32)
    vel = np.array([v1, v2], np.float32)
    u = np.array([u1, u2], np.float32)
    h = np.array([h1, h2], np.float32)
    return pos, vel, u, h


def perfect_lattice(n_side: int) -> np.ndarray:
    d = 1.0 / n_side
    g = (np.arange(n_side) + 0.5) * d
    zz, yy, xx = np.meshgrid(g, g, g, indexing="ij")
    return np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1).astype(np.float32)
