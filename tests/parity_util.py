"""Helpers of the GPU parity tests: run the CUDA path through the C ABI binding, run the oracle,
compare with the protocol of DESIGN.md "Parity protocol"."""
from __future__ import annotations

import numpy as np
import torch

from oracle import sph_oracle as O
from paper_2003_10850_b200 import binding as B

RTOL_RHO = 1e-5    # north_star: density and h within 1e-5 relative
RTOL_FORCE = 1e-4  # north_star: acceleration and du/dt within 1e-4 relative
FLOOR = 1e-3       # DESIGN.md R15: |a| is compared against max(|a|, FLOOR * sum_j |pair term|)
FLOOR_E2E = 1.0    # DESIGN.md R15c: end-to-end force (each side's own H, rho, Omega, equal only to 1e-5)
ULPS = 16          # DESIGN.md R15: fp32 resolution of a sum of pair terms, ULPS * 2^-24 * sqrt(sum_j term_j^2)
EDGE_MAX = 0.02    # upper bound on the edge-class fraction of an end-to-end density comparison


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


class GpuRun:
    """One context + device arrays for a ParticleSet-like input."""

    def __init__(self, pos, kernel, mass_scalar, box=1.0, mass=None, count_mode=0, max_iter=64, alpha=1.0, group_cap=0, group_node=0):
        self.n = pos.shape[0]
        self.sph = B.Sph(kernel=kernel, box=box, count_mode=count_mode, max_iter=max_iter, alpha_visc=alpha,
                         group_cap=group_cap, group_node=group_node)
        self.pos = dev(pos, torch.float32)
        self.mass = None if mass is None else dev(mass, torch.float32)
        self.sph.sph_build_index(self.pos, self.mass, mass_scalar)

    def density(self, h_guess, n_target, n_tol, active=None):
        n = self.n
        h = dev(h_guess, torch.float32).clone()
        rho = torch.full((n,), -1.0, device="cuda")
        om = torch.full((n,), -1.0, device="cuda")
        ngb = torch.full((n,), -1, device="cuda", dtype=torch.int32)
        st = torch.full((n,), -1, device="cuda", dtype=torch.int32)
        act = None if active is None else dev(active, torch.int32)
        unconv = self.sph.sph_density(h, rho, om, ngb, n_target, n_tol, active=act, status=st)
        torch.cuda.synchronize()
        return dict(H=h.cpu().numpy(), rho=rho.cpu().numpy(), omega=om.cpu().numpy(), Nint=ngb.cpu().numpy(),
                    status=st.cpu().numpy(), unconv=unconv)

    def force(self, vel, u, h, rho, omega, active=None):
        n = self.n
        acc = torch.full((n, 3), 7.0, device="cuda")
        du = torch.full((n,), 7.0, device="cuda")
        vs = torch.full((n,), 7.0, device="cuda")
        act = None if active is None else dev(active, torch.int32)
        self.sph.sph_hydro_force(dev(vel, torch.float32), dev(u, torch.float32), dev(h, torch.float32),
                                 dev(rho, torch.float32), dev(omega, torch.float32), acc, du, vs, active=act)
        torch.cuda.synchronize()
        return dict(acc=acc.cpu().numpy(), dudt=du.cpu().numpy(), vsig=vs.cpu().numpy())

    def close(self):
        self.sph.close()


def check_density_stage(g, o, sel=None, label=""):
    """Single evaluation at a common H: N_int bit-exact except oracle-flagged edge particles
    (a neighbour within 1e-6 relative of the support radius: counted, reported), rho/omega to 1e-5."""
    idx = slice(None) if sel is None else sel
    gn, grho, gom = g["Nint"][idx], g["rho"][idx].astype(np.float64), g["omega"][idx].astype(np.float64)
    edge = (o["edge"] & O.E_RADIUS) != 0
    mism = gn != o["Nint"]
    assert not np.any(mism & ~edge), f"{label}: N_int mismatch on non-edge particles: {np.flatnonzero(mism & ~edge)[:10]}"
    assert np.all(np.abs(gn[mism].astype(np.int64) - o["Nint"][mism]) <= 2)
    rel = np.abs(grho - o["rho"]) / o["rho"]
    assert rel.max() <= RTOL_RHO, f"{label}: rho rel err {rel.max():.3e}"
    om_o = o["omega"]
    # Omega: plain 1e-5 relative (north_star).  Only where Omega = 1 - D/(3S) has cancelled to |Omega| < 0.5
    # (arbitrary, unconverged H of the randomised sets; exactly 0 for a lone particle) is its error measured
    # against the magnitude of the terms that cancel, 1 + |1 - Omega| (R15b)
    small = np.abs(om_o) < 0.5
    relo = np.where(small, np.abs(gom - om_o) / (1.0 + np.abs(1.0 - om_o)), np.abs(gom - om_o) / np.maximum(np.abs(om_o), 0.5))
    assert relo.max() <= RTOL_RHO, f"{label}: omega err {relo.max():.3e}"
    return dict(n_edge=int(edge.sum()), n_mismatch=int(mism.sum()), rho_err=float(rel.max()), omega_err=float(relo.max()))


def check_density_e2e(g, o, ps_pos, h_guess, kernel, mass_scalar, n_target, n_tol, count_mode=0, sel=None, label="",
                      box=1.0, mass=None, edge_max=EDGE_MAX):
    """End-to-end iteration parity: non-edge particles H, rho to 1e-5 and N_int exact; edge-class
    particles are counted and checked conditionally (oracle re-evaluated at the GPU's H)."""
    idx = np.arange(len(g["H"])) if sel is None else np.asarray(sel)
    gH, grho, gn = g["H"][idx].astype(np.float64), g["rho"][idx].astype(np.float64), g["Nint"][idx]
    edge = o["edge"] != 0
    # the edge classes excuse a particle from the strict comparison: they must stay rare, or the test is hollow
    assert edge_max is None or edge.mean() <= edge_max or edge.sum() <= 2, f"{label}: edge-class fraction {edge.mean():.4f} > {edge_max}"
    relH = np.abs(gH - o["H"]) / o["H"]
    relr = np.abs(grho - o["rho"]) / o["rho"]
    ok = (relH <= RTOL_RHO) & (relr <= RTOL_RHO) & (gn == o["Nint"])
    bad = ~ok & ~edge
    # a disagreement on a non-edge particle is a failure ...
    assert not np.any(bad), (f"{label}: {bad.sum()} non-edge particles differ; worst H {relH[bad].max():.2e} "
                             f"rho {relr[bad].max():.2e}; ids {idx[bad][:8]}")
    # ... on an edge particle the GPU took the other branch: its own answer must still be a valid one
    chk = np.flatnonzero(~ok & edge)
    n_cond = len(chk)
    if n_cond:
        hh = np.array(h_guess, np.float32, copy=True)
        hh[idx[chk]] = g["H"][idx[chk]]
        e = O.density_eval(ps_pos, hh, kernel=kernel, mass_scalar=mass_scalar, mass=mass, box=box,
                           active=idx[chk].astype(np.int32))
        N = e["Nint"].astype(np.float64) if count_mode else e["Nw"]
        st = g["status"][idx[chk]]
        conv = (st & (1 << 8)) != 0
        assert np.all(np.abs(N[conv] - n_target) <= n_tol + 1e-4 * n_target), f"{label}: edge particle outside the band"
        assert np.all(np.abs(grho[chk] - e["rho"]) <= RTOL_RHO * e["rho"])
        mm = gn[chk] != e["Nint"]
        assert np.all(e["edge"][mm] != 0)
    return dict(n_edge=int(edge.sum()), edge_fraction=float(edge.mean()), n_conditional=int(n_cond), H_err=float(relH[ok].max() if ok.any() else 0),
                rho_err=float(relr[ok].max() if ok.any() else 0))


def untainted(pos, H, edge, box=1.0):
    """Particles that are not edge class and have no edge-class particle among their force neighbours
    (r < max(H_i, H_j), with a margin): the set on which an end-to-end force comparison is meaningful."""
    from scipy.spatial import cKDTree
    ok = ~edge
    ids = np.flatnonzero(edge)
    if len(ids) == 0:
        return ok
    P = np.mod(pos.astype(np.float64), box)
    tree = cKDTree(P, boxsize=box)
    etree = cKDTree(P[ids], boxsize=box)
    for lst in tree.query_ball_point(P[ids], r=H[ids] * 1.001):  # particles inside an edge particle's support
        ok[lst] = False
    hit = etree.query_ball_point(P, r=H * 1.001, return_length=True)  # edge particles inside a particle's support
    ok &= hit == 0
    return ok


def check_force(g, o, sel=None, label="", skip_vsig_edge=True, floor=FLOOR, mask=None):
    idx = slice(None) if sel is None else sel
    ga, gd, gv = g["acc"][idx].astype(np.float64), g["dudt"][idx].astype(np.float64), g["vsig"][idx].astype(np.float64)
    amag = np.sqrt((o["acc"] ** 2).sum(1))
    res = ULPS * 2.0 ** -24
    tol_a = RTOL_FORCE * np.maximum(amag, floor * o["asum"]) + res * np.sqrt(o["asq"])
    err_a = np.sqrt(((ga - o["acc"]) ** 2).sum(1))
    tol_a = np.where(tol_a > 0, tol_a, 1e-30)
    if mask is not None:  # compare only the particles selected by the mask
        tol_a = np.where(mask, tol_a, np.inf)
    assert np.all(err_a <= tol_a), f"{label}: acc err/tol max {np.max(err_a / tol_a):.3f} at {np.argmax(err_a / tol_a)}"
    tol_d = RTOL_FORCE * np.maximum(np.abs(o["dudt"]), floor * o["dusum"]) + res * np.sqrt(o["dusq"])
    tol_d = np.where(tol_d > 0, tol_d, 1e-30)
    if mask is not None:
        tol_d = np.where(mask, tol_d, np.inf)
    err_d = np.abs(gd - o["dudt"])
    wd = int(np.argmax(err_d / tol_d))
    assert np.all(err_d <= tol_d), (f"{label}: dudt err/tol max {np.max(err_d / tol_d):.3f} at {wd}: npair {o['npair'][wd]} "
                                    f"dudt {o['dudt'][wd]:.3e} dusum {o['dusum'][wd]:.3e} err {err_d[wd]:.3e}")
    edge = o["edge"] != 0
    relv = np.abs(gv - o["vsig"]) / np.maximum(o["vsig"], 1e-30)
    relv = np.where(o["vsig"] == 0, np.abs(gv), relv)
    m = ~edge if skip_vsig_edge else np.ones_like(edge)
    if mask is not None:
        m = m & mask
    assert np.all(relv[m] <= RTOL_RHO), f"{label}: vsig rel err {relv[m].max():.3e}"
    return dict(acc_err_over_tol=float(np.max(err_a / tol_a)), acc_relerr_max=float(np.max(err_a / np.maximum(amag, 1e-300))),
                dudt_err_over_tol=float(np.max(err_d / tol_d)), vsig_err=float(relv[m].max() if m.any() else 0),
                n_edge=int(edge.sum()))
