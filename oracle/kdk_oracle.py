"""Kick-drift-kick driver with power-of-two time bins -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain numpy (fp64) statement of reading R22 of DESIGN.md, on top of the oracle's density and
hydro-force functions.  The paper says only that Gadget3 "uses an adaptive time-stepping scheme" whose active
lists shrink to "one or very few" particles (PAPER.md:37 §1, :84-86 §2.2, :114 §3); the scheme below is the
kick-drift-kick integrator of the Gadget lineage [2], restated from its published description:

  timeline  T = 2^(n_bins-1) ticks per dt_max, tick length delta = dt_max / T; a particle of bin b steps
            s_b = T >> b ticks;
  criterion dt_i = min(courant * H_i / vsig_i, sqrt(2 eta H_i / |a_i|)); bin = smallest b with dt_max / 2^b <= dt_i,
            clamped to [0, n_bins - 1]; a longer step only one bin at a time and only where t % s_(b-1) == 0;
  init      density + force for all; bins; first half kick v += a s delta / 2, u += du/dt s delta / 2;
  step      t1 = t + (T >> max_i b_i); drift all: x += v (t1 - t) delta (periodic wrap);
            drifted v, u of everybody for the force pass: v + a tau, u + du/dt tau, tau = time since the middle of
            the particle's step; active = {i : t1 - tbegin_i == s_i}; density (last h as the guess) and force for the
            active particles; second half kick of the old step, new bin, first half kick of the new step.
  gravity   (optional, gravity = dict(G, r_s, r_cut, eps)): a_i = hydro force + the short-range gravity of R23 (direct
            sum) wherever the hydro force is evaluated; the time-step criterion sees the total acceleration.

Only tests/ may import this module; it imports nothing of the CUDA path.
"""
from __future__ import annotations

import numpy as np

from oracle import sph_oracle as O

F32 = np.float32


def new_bin(dt_max, n_bins, courant, eta, H, vsig, acc):
    """(bin, edge): edge marks particles whose log2(dt_max / dt) lies within 1e-4 of an integer (an fp32 evaluation may
    round to the other bin)."""
    a = np.sqrt((acc ** 2).sum(1))
    with np.errstate(divide="ignore", invalid="ignore"):
        dt = np.where(vsig > 0, courant * H / vsig, np.inf)
        dt = np.where(a > 0, np.minimum(dt, np.sqrt(2 * eta * H / a)), dt)
        x = np.log2(dt_max / dt)
    b = np.where(x > 0, np.ceil(x), 0).astype(np.int64)
    xf = np.where(np.isfinite(x), x, 0.5)
    edge = np.isfinite(x) & (np.abs(xf - np.round(xf)) < 1e-4) & (xf > -0.5) & (xf < n_bins - 0.5)
    return np.clip(b, 0, n_bins - 1).astype(np.int32), edge


def _grav(pos32, gravity, mass_scalar, box, active=None):
    """(acc, asum) of the short-range gravity for the active particles; zeros without gravity."""
    na = len(pos32) if active is None else len(active)
    if not gravity:
        return np.zeros((na, 3)), np.zeros(na)
    g = O.gravity_short(pos32, G=gravity["G"], r_s=gravity["r_s"], r_cut=gravity["r_cut"], eps=gravity["eps"], box=box,
                        mass_scalar=mass_scalar, active=active)
    return g["acc"], g["asum"]


def init(state, *, kernel, mass_scalar, dt_max, n_bins, n_ngb_target, n_ngb_tol, courant=0.3, eta=0.025, box=1.0, gravity=None):
    """state: dict with pos (n,3), vel (n,3), u, h (guess) as float arrays.  Returns the full state at tick 0 (fp64)."""
    pos = np.asarray(state["pos"], F32)
    n = len(pos)
    d = O.density(pos, np.asarray(state["h"], F32), kernel=kernel, n_target=n_ngb_target, n_tol=n_ngb_tol, mass_scalar=mass_scalar, box=box)
    f = O.hydro_force(pos, np.asarray(state["vel"], F32), np.asarray(state["u"], F32), d["H"].astype(F32), d["rho"].astype(F32),
                      d["omega"].astype(F32), kernel=kernel, mass_scalar=mass_scalar, box=box)
    T = 1 << (n_bins - 1)
    delta = dt_max / T
    ga, _ = _grav(pos, gravity, mass_scalar, box)
    f["acc"] = f["acc"] + ga
    b, edge = new_bin(dt_max, n_bins, courant, eta, d["H"], f["vsig"], f["acc"])
    hk = 0.5 * (T >> b) * delta
    out = dict(pos=pos.astype(np.float64), vel=np.asarray(state["vel"], np.float64) + f["acc"] * hk[:, None],
               u=np.asarray(state["u"], np.float64) + f["dudt"] * hk, h=d["H"], rho=d["rho"], omega=d["omega"], ngb=d["Nint"],
               acc=f["acc"], dudt=f["dudt"], vsig=f["vsig"], bin=b, tbegin=np.zeros(n, np.int32), tick=0, edge=edge)
    return out


def step(s, *, kernel, mass_scalar, dt_max, n_bins, n_ngb_target, n_ngb_tol, courant=0.3, eta=0.025, box=1.0, gravity=None):
    """One step from state s (as returned by init/step, or the GPU's state converted to numpy).  Returns the new state
    plus active (ids), vpred, upred, edge (bin decision within 1e-4 of switching, active particles only)."""
    T = 1 << (n_bins - 1)
    delta = dt_max / T
    b0 = np.asarray(s["bin"], np.int64)
    sstep = T >> b0
    ds = T >> int(b0.max())
    t1 = int(s["tick"]) + ds
    pos = np.asarray(s["pos"], np.float64) + np.asarray(s["vel"], np.float64) * (ds * delta)
    pos = np.where(pos >= box, pos - box, pos)
    pos = np.where(pos < 0, pos + box, pos)
    pos32 = pos.astype(F32)
    pos32 = np.where(pos32 >= F32(box), F32(0), pos32)
    tau = ((t1 - np.asarray(s["tbegin"], np.int64)) - 0.5 * sstep) * delta
    vpred = np.asarray(s["vel"], np.float64) + np.asarray(s["acc"], np.float64) * tau[:, None]
    upred = np.maximum(np.asarray(s["u"], np.float64) + np.asarray(s["dudt"], np.float64) * tau, 0.0)
    active = np.flatnonzero((t1 - np.asarray(s["tbegin"], np.int64)) == sstep).astype(np.int32)
    h = np.asarray(s["h"], np.float64).copy()
    rho = np.asarray(s["rho"], np.float64).copy()
    om = np.asarray(s["omega"], np.float64).copy()
    ngb = np.asarray(s["ngb"]).copy()
    d = O.density(pos32, h.astype(F32), kernel=kernel, n_target=n_ngb_target, n_tol=n_ngb_tol, mass_scalar=mass_scalar, box=box,
                  active=active)
    h[active], rho[active], om[active], ngb[active] = d["H"], d["rho"], d["omega"], d["Nint"]
    f = O.hydro_force(pos32, vpred.astype(F32), upred.astype(F32), h.astype(F32), rho.astype(F32), om.astype(F32), kernel=kernel,
                      mass_scalar=mass_scalar, box=box, active=active)
    acc = np.asarray(s["acc"], np.float64).copy()
    dudt = np.asarray(s["dudt"], np.float64).copy()
    vsig = np.asarray(s["vsig"], np.float64).copy()
    ga, gsum = _grav(pos32, gravity, mass_scalar, box, active=active)
    acc[active], dudt[active], vsig[active] = f["acc"] + ga, f["dudt"], f["vsig"]
    bn, edge = new_bin(dt_max, n_bins, courant, eta, h[active], vsig[active], acc[active])
    bo = b0[active]
    longer = bn < bo
    aligned = (t1 % np.maximum(T >> np.maximum(bo - 1, 0), 1)) == 0
    bn = np.where(longer, np.where(aligned, bo - 1, bo), bn).astype(np.int32)
    hk = 0.5 * ((T >> bo) + (T >> bn.astype(np.int64))) * delta
    vel = np.asarray(s["vel"], np.float64).copy()
    u = np.asarray(s["u"], np.float64).copy()
    vel[active] += acc[active] * hk[:, None]
    u[active] = np.maximum(u[active] + dudt[active] * hk, 0.0)
    b = np.asarray(s["bin"], np.int32).copy()
    tb = np.asarray(s["tbegin"], np.int32).copy()
    b[active] = bn
    tb[active] = t1
    return dict(pos=pos32.astype(np.float64), vel=vel, u=u, h=h, rho=rho, omega=om, ngb=ngb, acc=acc, dudt=dudt, vsig=vsig, bin=b,
                tbegin=tb, tick=t1, active=active, vpred=vpred, upred=upred, edge=edge, dens_edge=d["edge"], asum=f["asum"] + gsum, dusum=f["dusum"],
                asq=f["asq"], dusq=f["dusq"])
