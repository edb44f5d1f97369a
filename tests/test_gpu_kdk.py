"""GPU parity of the kick-drift-kick driver (sph_kdk_init / sph_kdk_step; R22) against the
oracle's driver, in lock step: every step of the GPU starts the oracle's step from the GPU's own previous state, so
rounding differences do not accumulate into different active lists; what is compared per step is the active list and
the bins (exact, except particles the oracle marks within 1e-4 of a bin boundary), positions, drifted and kicked
velocities and energies, and the hot-path outputs of the active particles."""
import numpy as np
import pytest
import torch

from oracle import kdk_oracle as K
from paper_2003_10850_b200 import binding as B
from paper_2003_10850_b200 import inputs as I

pytestmark = pytest.mark.gpu
F = ("pos", "vel", "u", "h", "rho", "omega", "ngb", "acc", "dudt", "vsig", "vpred", "upred", "bin", "tbegin", "active")


def _alloc(ps, h):
    n = ps.n
    z = lambda *s, dt=torch.float32: torch.zeros(*s, device="cuda", dtype=dt)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()
    return dict(pos=t(ps.pos), vel=t(ps.vel), u=t(ps.u), h=t(h), rho=z(n), omega=z(n), ngb=z(n, dt=torch.int32), acc=z(n, 3), dudt=z(n),
                vsig=z(n), vpred=z(n, 3), upred=z(n), bin=z(n, dt=torch.int32), tbegin=z(n, dt=torch.int32), active=z(n, dt=torch.int32))


def _np(st, tick):
    d = {k: st[k].cpu().numpy().astype(np.float64 if st[k].dtype == torch.float32 else np.int32) for k in F}
    d["tick"] = tick
    return d


def _close(a, b, rtol, scale, what):
    err = np.abs(np.asarray(a, np.float64) - np.asarray(b, np.float64))
    tol = rtol * np.maximum(np.abs(b), scale)
    assert np.all(err <= tol), f"{what}: worst err/tol {np.max(err / tol):.3f}"


# refresh_max = 0: an index build every step; 4 with rebuild_fraction 2: four refreshed steps (sph_refresh_index: the old
# tree with enlarged cells), then a rebuild, whatever the number of active particles -- the same results either way
# gravity: the short-range gravity of R23 added to the hydro acceleration (opening angle 0: the oracle's direct sum)
GRAV = dict(G=2.0, r_s=0.02, r_cut=0.09, eps=0.002, theta=0.0)


@pytest.mark.parametrize("shape,refresh_max,gravity", [("C1", 0, None), ("C1", 4, None), ("C3", 0, None), ("C3", 4, None), ("C3", 4, GRAV),
                                                       ("C1", 0, GRAV), ("C4", 4, None)])
def test_kdk_driver_in_lock_step_with_the_oracle(shape, refresh_max, gravity):
    if shape == "C1":
        ps = I.config1(12)
        rng = np.random.default_rng(9)
        ps.vel[:] = (0.2 * rng.normal(size=ps.vel.shape)).astype(np.float32)
        kw = dict(kernel=0, mass_scalar=ps.mass, dt_max=0.1, n_bins=5, n_ngb_target=64.0, n_ngb_tol=2.0)
        h0 = ps.h_guess
    elif shape == "C3":
        ps = I.config3(6000, 3)
        kw = dict(kernel=0, mass_scalar=ps.mass, dt_max=0.004, n_bins=8, n_ngb_target=64.0, n_ngb_tol=2.0)
        h0 = ps.h_guess
    else:  # the headline configuration's shape: NFW haloes, Wendland C6, 295 neighbours
        ps = I.config4(24000, 6, m_lo=320, m_hi=8000)
        kw = dict(kernel=ps.kernel, mass_scalar=ps.mass, dt_max=0.004, n_bins=8, n_ngb_target=ps.n_ngb, n_ngb_tol=ps.n_tol)
        h0 = ps.h_guess
    n = ps.n
    sph = B.Sph(kernel=kw["kernel"])
    st = _alloc(ps, h0)
    sph.sph_kdk_init(st, ps.mass, kw["dt_max"], kw["n_bins"], kw["n_ngb_target"], kw["n_ngb_tol"], refresh_max=refresh_max,
                     rebuild_fraction=2.0, gravity=gravity)
    if gravity:
        kw["gravity"] = {k: gravity[k] for k in ("G", "r_s", "r_cut", "eps")}
    torch.cuda.synchronize()
    g = _np(st, 0)
    o = K.init(dict(pos=ps.pos, vel=ps.vel, u=ps.u, h=h0), **kw)
    ok = ~o["edge"]
    assert np.array_equal(g["bin"][ok], o["bin"][ok]) and o["edge"].mean() < 0.01
    if gravity:  # gravity really takes part: the accelerations are those of the oracle with gravity, not without
        o0 = K.init(dict(pos=ps.pos, vel=ps.vel, u=ps.u, h=h0), **{**kw, "gravity": None})
        amax = np.abs(o["acc"]).max()
        assert np.abs(g["acc"] - o0["acc"]).max() > 1e-2 * amax and np.abs(g["acc"] - o["acc"]).max() < 1e-4 * amax
    vs = np.abs(o["vel"]).max()
    _close(g["vel"], o["vel"], 2e-4, 1e-3 * vs, "init vel")
    _close(g["u"], o["u"], 1e-4, 1e-3, "init u")
    nact, nbins = [], set()
    for step in range(10 if shape != "C4" else 6):
        tick, na = sph.sph_kdk_step(st, ps.mass)
        torch.cuda.synchronize()
        o = K.step(g, **kw)          # the oracle's step from the GPU's previous state
        g1 = _np(st, tick)
        assert tick == o["tick"] and na == len(o["active"]), (step, tick, o["tick"], na, len(o["active"]))
        a = o["active"]
        assert np.array_equal(g1["active"][:na], a)
        # drift: fp32 fma against fp64 + rounding
        d = np.abs(g1["pos"] - o["pos"])
        assert np.max(np.minimum(d, 1.0 - d)) < 2.5e-7
        _close(g1["vpred"], o["vpred"], 1e-5, 1e-3 * vs, "vpred")
        _close(g1["upred"], o["upred"], 1e-5, 1e-3, "upred")
        # hot path on the active particles (density end to end from the last h, force with the drifted state)
        de = o["dens_edge"] != 0
        assert de.mean() < 0.03
        _close(g1["h"][a][~de], o["h"][a][~de], 1e-5, 0.0, "h")
        _close(g1["rho"][a][~de], o["rho"][a][~de], 1e-5, 0.0, "rho")
        assert np.array_equal(g1["ngb"][a][~de], o["ngb"][a][~de])
        clean = np.ones(n, bool); clean[a[de]] = False  # (a diverged edge particle spoils its neighbours' force; rare: compare loosely)
        amag = np.sqrt((o["acc"][a] ** 2).sum(1))
        tol_a = 1e-4 * np.maximum(amag, o["asum"]) + 1e-6 * amag.max()
        assert np.all(np.sqrt(((g1["acc"][a] - o["acc"][a]) ** 2).sum(1)) <= tol_a)
        tol_d = 1e-4 * np.maximum(np.abs(o["dudt"][a]), o["dusum"]) + 1e-6 * np.abs(o["dudt"]).max()
        assert np.all(np.abs(g1["dudt"][a] - o["dudt"][a]) <= tol_d)
        # kicks and bins
        be = np.zeros(n, bool); be[a] = o["edge"]
        assert np.array_equal(g1["bin"][~be], o["bin"][~be]) and np.array_equal(g1["tbegin"], o["tbegin"])
        hk = 0.5 * (((1 << (kw["n_bins"] - 1)) >> g["bin"][a].astype(np.int64)) + ((1 << (kw["n_bins"] - 1)) >> o["bin"][a].astype(np.int64))) * kw["dt_max"] / (1 << (kw["n_bins"] - 1))
        okk = ~be[a]
        assert np.all(np.abs(g1["vel"][a] - o["vel"][a]).max(1)[okk] <= (hk * tol_a)[okk] + 2e-6 * vs)
        inact = np.ones(n, bool); inact[a] = False
        assert np.array_equal(g1["vel"][inact], g["vel"][inact]) and np.array_equal(g1["acc"][inact], g["acc"][inact])
        nact.append(na); nbins |= set(np.unique(g1["bin"]).tolist())
        g = g1
    print(shape, "kdk: active per step", nact, "bins", sorted(nbins))
    if shape in ("C3", "C4"):
        assert len(nbins) >= 3 and min(nact) < n // 4  # several bins, small active lists
    sph.close()
