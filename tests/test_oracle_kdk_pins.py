"""Pins of the oracle's kick-drift-kick driver (oracle/kdk_oracle.py; R22): closed forms
and invariants of the scheme, not the driver's own output."""
import math

import numpy as np

from oracle import kdk_oracle as K
from paper_2003_10850_b200 import inputs as I

G = 5.0 / 3.0


def test_lattice_at_rest_stays_at_rest_with_the_courant_bin():
    """Perfect lattice, v = 0, u = 1: no force, v_sig = 2 c for everybody, so dt = C H / (2 c) for everybody -- the bin
    follows by hand, every particle is active on every step, nothing ever moves."""
    n_side = 8
    pos = I.perfect_lattice(n_side)
    n = len(pos)
    H0 = 2.48232 / n_side
    st = dict(pos=pos, vel=np.zeros((n, 3), np.float32), u=np.ones(n, np.float32), h=np.full(n, H0 * 1.03, np.float32))
    kw = dict(kernel=0, mass_scalar=1.0 / n, dt_max=0.05, n_bins=6, n_ngb_target=64.0, n_ngb_tol=1e-3)
    s = K.init(st, **kw)
    c = math.sqrt(G * (G - 1))
    dt = 0.3 * H0 / (2 * c)
    b = math.ceil(math.log2(0.05 / dt))
    assert np.all(s["bin"] == b) and abs(s["h"].mean() / H0 - 1) < 1e-4
    assert np.max(np.abs(s["acc"])) < 1e-9 and np.max(np.abs(s["dudt"])) < 1e-12
    tick = 0
    for _ in range(3):
        s = K.step(s, **kw)
        tick += (1 << 5) >> b
        assert s["tick"] == tick and len(s["active"]) == n and np.all(s["bin"] == b)
        assert np.array_equal(s["pos"], pos.astype(np.float64)) and np.max(np.abs(s["vel"])) < 1e-9


def test_free_streaming_and_periodic_wrap():
    """Two particles out of each other's reach feel nothing (no neighbour: a = 0, v_sig = 0, dt = infinity, bin 0):
    x(t) = x0 + v t through the periodic wall, exactly as the drift says."""
    pos = np.array([[0.9, 0.5, 0.5], [0.3, 0.1, 0.2]], np.float32)
    vel = np.array([[0.8, 0.0, -0.4], [-0.6, 0.2, 0.0]], np.float32)
    st = dict(pos=pos, vel=vel, u=np.ones(2, np.float32), h=np.full(2, 0.1, np.float32))
    kw = dict(kernel=0, mass_scalar=1.0, dt_max=0.125, n_bins=4, n_ngb_target=1.0, n_ngb_tol=10.0)
    s = K.init(st, **kw)
    assert np.all(s["bin"] == 0) and np.all(s["acc"] == 0) and np.all(s["vsig"] == 0)
    for k in range(1, 5):
        s = K.step(s, **kw)
        want = np.mod(pos.astype(np.float64) + vel.astype(np.float64) * 0.125 * k, 1.0)
        d = np.abs(s["pos"] - want)
        assert s["tick"] == 8 * k and np.max(np.minimum(d, 1.0 - d)) < 2e-7  # (positions are handed on in fp32; periodic distance)
        assert np.array_equal(s["vel"], vel.astype(np.float64))


def _energy(s, m, T, delta):
    """Total energy and momentum at the synchronisation point: undo the first half kick of the step just opened."""
    hk = 0.5 * (T >> s["bin"].astype(np.int64)) * delta
    v = s["vel"] - s["acc"] * hk[:, None]
    u = s["u"] - s["dudt"] * hk
    return m * (0.5 * (v ** 2).sum() + u.sum()), m * v.sum(0)


def test_fixed_step_kdk_conserves_momentum_and_is_second_order():
    """One bin (n_bins = 1): everybody steps dt_max, the scheme is the plain leapfrog.  Momentum is conserved to rounding
    at every step (all active, antisymmetric pair terms); the energy error over a fixed time span falls by ~4 when the
    step is halved (second order)."""
    ps = I.config1(6)
    rng = np.random.default_rng(2)
    n = ps.n
    vel = (0.05 * rng.normal(size=(n, 3))).astype(np.float32)
    errs = []
    for dt in (0.02, 0.01):
        st = dict(pos=ps.pos, vel=vel, u=ps.u, h=ps.h_guess)
        kw = dict(kernel=0, mass_scalar=ps.mass, dt_max=dt, n_bins=1, n_ngb_target=ps.n_ngb, n_ngb_tol=0.05)
        s = K.init(st, **kw)
        e0, p0 = _energy(s, ps.mass, 1, dt)
        for _ in range(round(0.08 / dt)):
            s = K.step(s, **kw)
            e, p = _energy(s, ps.mass, 1, dt)
            assert np.all(np.abs(p - p0) < 1e-9 * ps.mass * np.abs(s["vel"]).sum())
        errs.append(abs(e - e0) / e0)
    assert errs[0] < 2e-4 and 2.5 < errs[0] / errs[1] < 6.5, errs


def test_time_bin_structure():
    """Over many steps of a clustered set: the timeline only moves forward to the next end of a step; a particle is
    active exactly when its own step ends; steps begin on multiples of their length; a bin may rise freely and falls by
    at most one at a time."""
    ps = I.config3(600, 2)
    kw = dict(kernel=0, mass_scalar=ps.mass, dt_max=0.02, n_bins=6, n_ngb_target=40.0, n_ngb_tol=1.0)
    s = K.init(dict(pos=ps.pos, vel=ps.vel, u=ps.u, h=ps.h_guess * 0.9), **kw)
    T = 1 << 5
    assert len(np.unique(s["bin"])) >= 3  # several bins occupied: the set is clustered
    nact = []
    for _ in range(24):
        b0, tb0, t0 = s["bin"].copy(), s["tbegin"].copy(), s["tick"]
        s = K.step(s, **kw)
        t1 = s["tick"]
        assert t1 == t0 + (T >> b0.max())
        ends = (t1 - tb0) == (T >> b0.astype(np.int64))
        assert np.array_equal(np.flatnonzero(ends), s["active"]) and len(s["active"]) >= 1
        assert np.all((t1 - tb0)[~ends] < (T >> b0.astype(np.int64))[~ends])      # nobody oversteps
        a = s["active"]
        assert np.all(s["tbegin"][a] == t1) and np.all(t1 % (T >> s["bin"][a].astype(np.int64)) == 0)
        assert np.all(s["bin"][a] >= b0[a] - 1)
        inact = np.ones(ps.n, bool); inact[a] = False
        assert np.array_equal(s["bin"][inact], b0[inact]) and np.array_equal(s["acc"][inact], s["acc"][inact])
        nact.append(len(a))
    assert min(nact) < ps.n // 2  # most steps update a part of the particles only (the paper's regime)


GRAV = dict(G=1.0, r_s=0.05, r_cut=0.225, eps=0.01)


def _grav_factor(r, g):
    """Closed form of R23 for one pair: G fac(r) / (r^2 + eps^2)^(3/2), fac = erfc(r / 2 r_s) + r / (r_s sqrt(pi)) exp(-r^2 / 4 r_s^2)."""
    x = r / (2 * g["r_s"])
    return g["G"] * (math.erfc(x) + r / (g["r_s"] * math.sqrt(math.pi)) * math.exp(-x * x)) / (r * r + g["eps"] ** 2) ** 1.5


def test_two_bodies_under_gravity_follow_the_leapfrog_by_hand():
    """Two gas particles outside each other's SPH support but inside r_cut: the only force is the short-range gravity of
    R23, known in closed form; with one bin the first step is x1 = x0 + v0 dt + a0 dt^2 / 2 exactly."""
    r = 0.125
    pos = np.array([[0.5 - r / 2, 0.5, 0.5], [0.5 + r / 2, 0.5, 0.5]], np.float32)
    st = dict(pos=pos, vel=np.zeros((2, 3), np.float32), u=np.ones(2, np.float32), h=np.full(2, 0.03, np.float32))
    m, dt = 0.25, 0.0625
    kw = dict(kernel=0, mass_scalar=m, dt_max=dt, n_bins=1, n_ngb_target=1.0, n_ngb_tol=10.0, gravity=GRAV)
    s = K.init(st, **kw)
    a0 = m * _grav_factor(r, GRAV) * r  # towards each other
    assert abs(s["acc"][0, 0] - a0) < 1e-12 * a0 and abs(s["acc"][1, 0] + a0) < 1e-12 * a0 and np.all(s["acc"][:, 1:] == 0)
    assert np.all(s["vsig"] == 0) and np.all(s["dudt"] == 0)  # no SPH neighbour
    s1 = K.step(s, **kw)
    assert abs(s1["pos"][0, 0] - (pos[0, 0] + 0.5 * a0 * dt * dt)) < 1e-7
    assert abs(s1["pos"][1, 0] - (pos[1, 0] - 0.5 * a0 * dt * dt)) < 1e-7
    r1 = float(s1["pos"][1, 0] - s1["pos"][0, 0])
    a1 = m * _grav_factor(r1, GRAV) * r1
    assert abs(s1["acc"][0, 0] - a1) < 1e-10 * a1 and a1 > a0  # closer, stronger
    # without the option nothing pulls
    s0 = K.init(st, **{**kw, "gravity": None})
    assert np.all(s0["acc"] == 0)


def test_gravity_in_the_driver_conserves_momentum_and_vanishes_on_the_lattice():
    ps = I.config1(6)
    rng = np.random.default_rng(4)
    vel = (0.05 * rng.normal(size=(ps.n, 3))).astype(np.float32)
    kw = dict(kernel=0, mass_scalar=ps.mass, dt_max=0.01, n_bins=1, n_ngb_target=ps.n_ngb, n_ngb_tol=0.05, gravity=dict(GRAV, G=50.0))
    s = K.init(dict(pos=ps.pos, vel=vel, u=ps.u, h=ps.h_guess), **kw)
    s_h = K.init(dict(pos=ps.pos, vel=vel, u=ps.u, h=ps.h_guess), **{**kw, "gravity": None})
    assert np.abs(s["acc"] - s_h["acc"]).max() > 0.05 * np.abs(s_h["acc"]).max()  # gravity takes part
    _, p0 = _energy(s, ps.mass, 1, 0.01)
    for _ in range(3):
        s = K.step(s, **kw)
        _, p = _energy(s, ps.mass, 1, 0.01)
        assert np.all(np.abs(p - p0) < 1e-9 * ps.mass * np.abs(s["vel"]).sum())
    # perfect lattice: every pair term has its mirror image, gravity cancels like the pressure force does
    n_side = 8
    pos = I.perfect_lattice(n_side)
    n = len(pos)
    st = dict(pos=pos, vel=np.zeros((n, 3), np.float32), u=np.ones(n, np.float32), h=np.full(n, 1.03 * 2.48232 / n_side, np.float32))
    s = K.init(st, kernel=0, mass_scalar=1.0 / n, dt_max=0.05, n_bins=6, n_ngb_target=64.0, n_ngb_tol=1e-3, gravity=GRAV)
    assert np.max(np.abs(s["acc"])) < 1e-9
