"""Pins of the improved-SPH extension of the oracle (R17-R20): values the mathematics
fixes -- isotropy of a cubic lattice, reductions to the separately pinned base force, two particles by hand,
conservation laws -- not the oracle's own output."""
import math

import numpy as np
import pytest

from oracle import sph_oracle as O
from paper_2003_10850_b200 import inputs as I

G = 5.0 / 3.0


def _lattice(n_side=12):
    pos = I.perfect_lattice(n_side)
    n = len(pos)
    H = np.full(n, 4.12941 / n_side, np.float32)  # Wendland C6, N_w = 295 (perfect-lattice pin of the base oracle)
    rho = np.full(n, 1.0, np.float32)
    centre = np.flatnonzero(np.all(np.abs(pos - 0.5) < 0.5 - float(H[0]) - 1.0 / n_side, axis=1)).astype(np.int32)
    assert len(centre) >= 8
    return pos, H, rho, centre


def test_velocity_gradients_on_a_cubic_lattice():
    """R17 on a linear field v = A (x - 1/2): on a cubic lattice sum_j f(r_j) d_j d_j^T is isotropic (t times the unit
    matrix), so div v = t tr A and curl v = t (A_zy - A_yz, A_xz - A_zx, A_yx - A_xy) with ONE factor t, which tends
    to 1 in the continuum (-int r dW/dr d^3r = 3 int W = 3).  A symmetric A has no curl, an antisymmetric one no
    divergence, a uniform velocity neither -- exactly."""
    pos, H, rho, act = _lattice()
    rng = np.random.default_rng(11)
    A = rng.normal(size=(3, 3))
    x = pos.astype(np.float64) - 0.5
    kw = dict(kernel=1, mass_scalar=1.0 / len(pos), active=act)

    def grad(M):
        return O.velocity_gradients(pos, (x @ M.T).astype(np.float32), H, rho, **kw)

    g = grad(A)
    om = np.array([A[2, 1] - A[1, 2], A[0, 2] - A[2, 0], A[1, 0] - A[0, 1]])
    t = g["divv"] / np.trace(A)
    assert np.ptp(t) < 2e-6 and abs(t.mean() - 1.0) < 0.01, (t.min(), t.max())  # (fp32 velocities: 1e-7 relative)
    assert np.max(np.abs(g["curlv"] - t.mean() * om)) < 1e-5 * np.abs(om).max()
    gs = grad(A + A.T)
    assert np.max(np.abs(gs["curlv"])) < 1e-5 and np.max(np.abs(gs["divv"] / (2 * np.trace(A)) - t.mean())) < 2e-6
    ga = grad(A - A.T)
    assert np.max(np.abs(ga["divv"])) < 1e-5
    v0 = np.tile(np.array([0.3, -1.0, 2.0], np.float32), (len(pos), 1))
    gu = O.velocity_gradients(pos, v0, H, rho, **kw)
    assert np.all(gu["divv"] == 0.0) and np.all(gu["curlv"] == 0.0)


def _random_state(n=600, seed=3):
    rng = np.random.default_rng(seed)
    pos = rng.uniform(0, 1, (n, 3)).astype(np.float32)
    vel = rng.normal(0, 0.3, (n, 3)).astype(np.float32)
    u = rng.uniform(0.5, 2.0, n).astype(np.float32)
    H = rng.uniform(0.15, 0.25, n).astype(np.float32)
    rho = rng.uniform(0.5, 2.0, n).astype(np.float32)
    om = rng.uniform(0.8, 1.2, n).astype(np.float32)
    return pos, vel, u, H, rho, om, 1.0 / n


@pytest.mark.parametrize("k", [0, 1])
def test_improved_force_reduces_to_the_base_force(k):
    """Constant alpha, no limiter, no conduction: R18-R20 drop out and the improved pair sum is the (separately pinned)
    base one.  With the limiter on and a shear-only velocity-gradient state (div v = 0, curl v != 0) f = 0 exactly:
    the viscosity is gone and the result is the base force at alpha = 0."""
    pos, vel, u, H, rho, om, m = _random_state()
    n = len(pos)
    a0 = 0.75  # (exact in fp32: alpha is an fp32 array on the improved side)
    al = np.full(n, a0, np.float32)
    dv, cv = np.zeros(n, np.float32), np.zeros((n, 3), np.float32)
    base = O.hydro_force(pos, vel, u, H, rho, om, kernel=k, mass_scalar=m, alpha=a0, brute=True)
    imp = O.hydro_force_improved(pos, vel, u, H, rho, om, al, dv, cv, kernel=k, mass_scalar=m, alpha_cond=0.0, balsara=False)
    for key in ("acc", "dudt", "vsig"):
        assert np.max(np.abs(imp[key] - base[key])) <= 1e-12 * np.max(np.abs(base[key]))
    cv[:, 2] = -1.3
    shear = O.hydro_force_improved(pos, vel, u, H, rho, om, al, dv, cv, kernel=k, mass_scalar=m, alpha_cond=0.0, balsara=True)
    inviscid = O.hydro_force(pos, vel, u, H, rho, om, kernel=k, mass_scalar=m, alpha=0.0, brute=True)
    assert np.max(np.abs(shear["acc"] - inviscid["acc"])) <= 1e-12 * np.max(np.abs(inviscid["acc"]))
    assert np.max(np.abs(shear["dudt"] - inviscid["dudt"])) <= 1e-12 * np.max(np.abs(inviscid["dudt"]))
    assert np.max(np.abs(shear["vsig"] - base["vsig"])) < 1e-14  # the signal velocity does not depend on alpha or f


def test_two_particles_by_hand():
    """Two approaching particles with different alpha, limiter values and internal energies: every factor of R18-R20
    written out by hand (kernel derivative from the pinned orc_dWdr)."""
    r, h1, h2 = 0.1, 0.25, 0.2
    pos, vel, u, H = I.two_particles(r, h1, h2, u1=1.5, u2=0.75, v1=(0.4, 0, 0), v2=(-0.2, 0, 0))
    rho = np.array([1.2, 0.9], np.float32)
    om = np.array([1.1, 0.95], np.float32)
    al = np.array([0.5, 1.5], np.float32)
    dv = np.array([-2.0, 0.5], np.float32)
    cv = np.array([[0, 0, 1.0], [0.5, 0, 0]], np.float32)
    m, ac, amin, amax, ell = 0.3, 0.25, 0.02, 3.0, 4.0
    o = O.hydro_force_improved(pos, vel, u, H, rho, om, al, dv, cv, kernel=1, mass_scalar=m, alpha_cond=ac, alpha_min=amin,
                               alpha_max=amax, decay_l=ell, balsara=True)
    rr = float(pos[1, 0]) - float(pos[0, 0])  # the fp32 separation the oracle sees
    uu, rh, oo, hh = u.astype(np.float64), rho.astype(np.float64), om.astype(np.float64), H.astype(np.float64)
    c = np.sqrt(G * (G - 1) * uu)
    P = (G - 1) * rh * uu
    A = (G - 1) * uu / (oo * rh)
    F = [O.dWdr(1, rr, hh[0]), O.dWdr(1, rr, hh[1])]
    f = [abs(float(dv[i])) / (abs(float(dv[i])) + float(np.linalg.norm(cv[i])) + 1e-4 * c[i] / hh[i]) for i in (0, 1)]
    # particle 0 sits at smaller x: rhat_01 = -x, v_01 . rhat = -(0.4 + 0.2) = -0.6 (approaching)
    vr = -(float(vel[0, 0]) - float(vel[1, 0]))
    mu = min(vr, 0.0)
    vs = c[0] + c[1] - 3 * mu
    rb = 0.5 * (rh[0] + rh[1])
    PI = -0.5 * 0.5 * (float(al[0]) + float(al[1])) * vs * mu / rb * 0.5 * (f[0] + f[1])
    Fb = 0.5 * (F[0] + F[1])
    t = m * (A[0] * F[0] + A[1] * F[1] + PI * Fb)
    assert abs(o["acc"][0, 0] - t) < 1e-12 * abs(t) and abs(o["acc"][1, 0] + t) < 1e-12 * abs(t)  # a_0 = -t rhat = +t x
    cond = m * ac * math.sqrt(abs(P[0] - P[1]) / rb) * (uu[0] - uu[1]) * Fb / rb
    assert cond < 0  # the hotter particle cools
    e0 = m * (A[0] * F[0] + 0.5 * PI * Fb) * vr + cond
    e1 = m * (A[1] * F[1] + 0.5 * PI * Fb) * vr - cond
    assert abs(o["dudt"][0] - e0) < 1e-12 * abs(e0) and abs(o["dudt"][1] - e1) < 1e-12 * abs(e1)
    assert abs(o["ducond"][0] - cond) < 1e-12 * abs(cond) and abs(o["ducond"][0] + o["ducond"][1]) < 1e-15
    assert abs(o["vsig"][0] - vs) < 1e-12
    # R19: d alpha/dt = -(alpha - alpha_min) 2 l c / H + max(0, -div v)(alpha_max - alpha)
    da0 = -(float(al[0]) - amin) * 2 * ell * c[0] / hh[0] + 2.0 * (amax - float(al[0]))
    da1 = -(float(al[1]) - amin) * 2 * ell * c[1] / hh[1]
    assert abs(o["dalpha"][0] - da0) < 1e-12 * abs(da0) and abs(o["dalpha"][1] - da1) < 1e-12 * abs(da1)


@pytest.mark.parametrize("k", [0, 1])
def test_improved_force_conserves_momentum_and_energy(k):
    """alpha_ij, f_ij, rho_ij and Fbar_ij are symmetric in i <-> j and the conduction term antisymmetric: with all
    particles active sum m a = 0 and sum m (v . a + du/dt) = 0 to rounding, and conduction alone moves no net energy."""
    pos, vel, u, H, rho, om, m = _random_state(500, 8)
    n = len(pos)
    rng = np.random.default_rng(1)
    al = rng.uniform(0.02, 3.0, n).astype(np.float32)
    dv = rng.normal(0, 2.0, n).astype(np.float32)
    cv = rng.normal(0, 2.0, (n, 3)).astype(np.float32)
    o = O.hydro_force_improved(pos, vel, u, H, rho, om, al, dv, cv, kernel=k, mass_scalar=m)
    a = o["acc"]
    assert np.all(np.abs(a.sum(0)) <= 1e-12 * np.abs(a).sum(0))
    e = (vel.astype(np.float64) * a).sum(1) + o["dudt"]
    assert abs(e.sum()) <= 1e-12 * (np.abs((vel.astype(np.float64) * a).sum(1)).sum() + o["dusum"].sum())
    assert abs(o["ducond"].sum()) <= 1e-13 * np.abs(o["ducond"]).sum() and np.abs(o["ducond"]).sum() > 0
    # conduction flows from hot to cold: on a static gas whose only structure is a step in u the hot side loses energy
    vel0 = np.zeros_like(vel)
    us = np.where(pos[:, 0] < 0.5, 2.0, 1.0).astype(np.float32)
    one = np.ones(n, np.float32)
    s = O.hydro_force_improved(pos, vel0, us, np.full(n, 0.2, np.float32), one, one, al, dv, cv, kernel=k, mass_scalar=m)
    assert np.all(s["ducond"][us > 1.5] <= 0) and np.all(s["ducond"][us < 1.5] >= 0) and s["ducond"].min() < 0


# ------------------------------------------------------------------ thermal conduction (R21)
def test_thermal_conduction_closed_forms_on_a_lattice():
    """R21 with a constant conductivity on a cubic lattice (rho = 1): a uniform temperature conducts nothing, a linear
    one neither (inversion symmetry: exactly), and T = x^2 gives du/dt = kappa lap(T) / rho = 2 kappa times the SAME
    isotropy factor t of the lattice that the velocity-gradient estimator has (R17 pin) -- two routines, one number.
    (16^3 lattice: coordinates, T and the velocities are dyadic rationals, exact in fp32.)"""
    pos, H, rho, act = _lattice(16)
    n = len(pos)
    m = 1.0 / n
    x = pos[:, 0].astype(np.float64) - 0.5
    kw = dict(kernel=1, kappa0=0.3, kappa_exp=0.0, mass_scalar=m, active=act)
    assert np.all(O.thermal_conduction(pos, np.full(n, 1.7, np.float32), H, rho, **kw)["dudt"] == 0.0)
    lin = O.thermal_conduction(pos, (2.0 + 0.5 * x).astype(np.float32), H, rho, **kw)
    assert np.max(np.abs(lin["dudt"])) < 1e-13 * lin["dusum"].max()
    quad = O.thermal_conduction(pos, (1.0 + x * x).astype(np.float32), H, rho, **kw)
    A = np.diag([1.0, 2.0, -0.5])
    t = O.velocity_gradients(pos, ((pos.astype(np.float64) - 0.5) @ A.T).astype(np.float32), H, rho, kernel=1, mass_scalar=m,
                             active=act)["divv"] / np.trace(A)
    assert np.max(np.abs(quad["dudt"] / (2 * 0.3) - t)) < 1e-7 and abs(t.mean() - 1) < 0.01  # (kappa0 = 0.3 is not dyadic)


def test_thermal_conduction_two_particles_and_conservation():
    r, h1, h2 = 0.1, 0.25, 0.2
    pos, vel, u, H = I.two_particles(r, h1, h2, u1=2.0, u2=0.5)
    rho = np.array([1.2, 0.9], np.float32)
    m, k0 = 0.3, 0.7
    o = O.thermal_conduction(pos, u, H, rho, kernel=1, kappa0=k0, kappa_exp=2.5, mass_scalar=m)
    rr = float(pos[1, 0]) - float(pos[0, 0])
    k = [k0 * 2.0 ** 2.5, k0 * 0.5 ** 2.5]
    Fb = 0.5 * (O.dWdr(1, rr, float(H[0])) + O.dWdr(1, rr, float(H[1])))
    e0 = m / (float(rho[0]) * float(rho[1])) * 4 * k[0] * k[1] / (k[0] + k[1]) * (2.0 - 0.5) * Fb / rr
    assert e0 < 0 and abs(o["dudt"][0] - e0) < 1e-12 * abs(e0) and abs(o["dudt"][1] + e0) < 1e-12 * abs(e0)  # hot cools, cold heats
    pos, vel, u, H, rho, om, m = _random_state(500, 4)
    o = O.thermal_conduction(pos, u, H, rho, kernel=0, kappa0=1.0, mass_scalar=m)
    assert abs(o["dudt"].sum()) < 1e-12 * o["dusum"].sum() and o["dusum"].sum() > 0  # equal masses: sum m du/dt = 0


# ------------------------------------------------------------------ short-range gravity (R23)
def test_gravity_short_two_particles_and_potential():
    """R23: two particles -- the closed form with math.erfc, its Newtonian limit for r << r_s, the force as minus the
    derivative of the short-range potential -G m erfc(r / 2 r_s) / r (finite difference), truncation at r_cut, and the
    pair through the periodic wall."""
    G, rs, m = 2.0, 0.05, 0.3
    for r in (0.003, 0.02, 0.07, 0.15):
        pos = np.array([[0.25, 0.5, 0.5], [0.25 + r, 0.5, 0.5]], np.float32)
        rr = float(pos[1, 0]) - float(pos[0, 0])
        o = O.gravity_short(pos, G=G, r_s=rs, r_cut=0.2, eps=0.0, mass_scalar=m)
        x = rr / (2 * rs)
        F = G * m / rr ** 2 * (math.erfc(x) + rr / (rs * math.sqrt(math.pi)) * math.exp(-x * x))
        assert abs(o["acc"][0, 0] - F) < 1e-12 * F and abs(o["acc"][1, 0] + F) < 1e-12 * F  # attraction, antisymmetric
        phi = lambda q: -G * m * math.erfc(q / (2 * rs)) / q
        h = 1e-6 * rr
        assert abs((phi(rr + h) - phi(rr - h)) / (2 * h) - F) < 1e-6 * F                      # F = -dPhi/dr (on particle 0: +x)
        if r == 0.003:
            assert abs(F / (G * m / rr ** 2) - 1) < 1e-4                                       # Newtonian for r << r_s
    far = np.array([[0.1, 0.5, 0.5], [0.35, 0.5, 0.5]], np.float32)
    assert np.all(O.gravity_short(far, G=G, r_s=rs, r_cut=0.2, eps=0.0, mass_scalar=m)["acc"] == 0)  # beyond r_cut
    wall = np.array([[0.02, 0.5, 0.5], [0.97, 0.5, 0.5]], np.float32)
    assert O.gravity_short(wall, G=G, r_s=rs, r_cut=0.2, eps=0.0, mass_scalar=m)["acc"][0, 0] < 0   # pulled through the wall
    soft = O.gravity_short(np.array([[0.5, 0.5, 0.5], [0.51, 0.5, 0.5]], np.float32), G=G, r_s=rs, r_cut=0.2, eps=0.02, mass_scalar=m)
    rr = float(np.float32(0.51)) - 0.5
    x = rr / (2 * rs)
    Fs = G * m * rr / (rr ** 2 + 0.02 ** 2) ** 1.5 * (math.erfc(x) + rr / (rs * math.sqrt(math.pi)) * math.exp(-x * x))
    assert abs(soft["acc"][0, 0] - Fs) < 1e-12 * Fs


def test_gravity_short_symmetries():
    """Momentum: sum m a = 0 to rounding (all active); a perfect lattice feels nothing (inversion symmetry)."""
    pos, vel, u, H, rho, om, m = _random_state(500, 12)
    o = O.gravity_short(pos, G=1.0, r_s=0.04, r_cut=0.18, eps=0.005, mass_scalar=m)
    assert np.all(np.abs(o["acc"].sum(0)) < 1e-12 * np.abs(o["acc"]).sum(0))
    lat = I.perfect_lattice(8)
    ol = O.gravity_short(lat, G=1.0, r_s=0.04, r_cut=0.18, eps=0.0, mass_scalar=1.0 / len(lat))
    assert np.max(np.abs(ol["acc"])) < 1e-12 * ol["asum"].max()
