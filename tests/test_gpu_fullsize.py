"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (library
defaults): the whole set goes through sph_build_index -> sph_density -> sph_hydro_force on the GPU, and
a seeded sample of particles is recomputed one by one by the fp64 oracle.
Density: end to end from the same guess.  Force: stage-isolated, the GPU's own converged (H, rho, Omega)
of ALL particles are the inputs of both sides (the sampled particles' neighbours need them)."""
import numpy as np
import pytest
import torch

from oracle import sph_oracle as O
from paper_2003_10850_b200 import binding as B
from paper_2003_10850_b200 import inputs as I
from parity_util import GpuRun, check_density_e2e, check_force

pytestmark = pytest.mark.gpu

SAMPLE = 4096
_cache = {}


def _stratified_sample(ps, pool, rng):
    """SAMPLE particle ids of the pool.  Sets with haloes (generator metadata aux["halo"], aux["radius"]) are
    sampled by strata of halo-centric radius -- background, then eight logarithmic bins of r / r_vir down to the
    cusps -- so that the deep octree levels and the cores of the largest haloes are represented; other sets
    uniformly."""
    aux = ps.aux
    if "halo" not in aux or "r_vir" not in aux:
        return np.sort(rng.choice(pool, min(SAMPLE, len(pool)), replace=False)).astype(np.int32)
    halo = aux["halo"][pool]
    x = np.where(halo >= 0, aux["radius"][pool] / aux["r_vir"][np.maximum(halo, 0)], np.inf)
    edges = np.concatenate([[0.0], np.logspace(-2.5, 0.0, 8)])
    strata = [pool[halo < 0]] + [pool[(halo >= 0) & (x > lo) & (x <= hi)] for lo, hi in zip(edges[:-1], edges[1:])]
    strata = [st for st in strata if len(st)]
    per = SAMPLE // len(strata)
    pick = [rng.choice(st, min(per, len(st)), replace=False) for st in strata]
    # the cores of the ten largest haloes: the deepest octree levels
    big = np.argsort(-aux["per"])[:10]
    core = pool[np.isin(halo, big) & (x <= edges[2])]
    if len(core):
        pick.append(rng.choice(core, min(per // 2, len(core)), replace=False))
    return np.unique(np.concatenate(pick)).astype(np.int32)


def _set(name):
    if name not in _cache:
        _cache.clear()  # one full-size set at a time in host memory
        _cache[name] = {"C2": I.config2, "C3": I.config3, "C4": I.config4}[name]()
    return _cache[name]


def _sampled_parity(ps, active_all, label):
    rng = np.random.default_rng(I.SEED_BASE + 77)
    pool = np.arange(ps.n, dtype=np.int32) if active_all is None else active_all
    sample = _stratified_sample(ps, pool, rng)
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    gd = g.density(ps.h_guess, ps.n_ngb, ps.n_tol, active=active_all)
    assert gd["unconv"] == 0
    st = g.sph.stats()
    n_act = ps.n if active_all is None else len(active_all)
    assert st["dens_evals"] >= n_act and st["dens_pairs"] > 30 * n_act
    # density end to end on the sample (oracle: same guess, same rule)
    o = O.density(ps.pos, ps.h_guess, kernel=ps.kernel, n_target=ps.n_ngb, n_tol=ps.n_tol, mass_scalar=ps.mass,
                  active=sample)
    rep = check_density_e2e(gd, o, ps.pos, ps.h_guess, ps.kernel, ps.mass, ps.n_ngb, ps.n_tol, sel=sample, label=label)
    # properties that hold at any size: every active converged inside the band; inactive entries untouched
    conv = (gd["status"] & B.ST_CONVERGED) != 0
    if active_all is None:
        assert conv.all() and np.all(gd["rho"] > 0) and np.all(gd["Nint"] >= 1)
    else:
        assert conv[active_all].all()
        inact = np.ones(ps.n, bool); inact[active_all] = False
        assert np.all(gd["rho"][inact] == -1)
    return g, gd, sample, rep


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_fullsize_all_active(name):
    ps = _set(name)
    g, gd, sample, rep = _sampled_parity(ps, None, name + " full e2e")
    H, rho, om = gd["H"], gd["rho"], gd["omega"]
    gf = g.force(ps.vel, ps.u, H, rho, om)
    of = O.hydro_force(ps.pos, ps.vel, ps.u, H, rho, om, kernel=ps.kernel, mass_scalar=ps.mass, active=sample)
    repf = check_force(gf, of, sel=sample, label=name + " full force")
    # momentum: all particles active => sum m a = 0 to rounding (pair terms antisymmetric)
    a = gf["acc"].astype(np.float64)
    assert np.all(np.abs(a.sum(0)) <= 1e-5 * np.abs(a).sum(0))
    print(name, "full", rep, repf, g.sph.stats())
    g.close()


def test_fullsize_extensions():
    """The SURVEY.md §8(f) pair passes at configs[3]'s full size (10^7 particles, library defaults): velocity gradients,
    improved force, thermal conduction and short-range gravity run over ALL particles on the GPU; the oracle's plain
    sums over all j recompute 256 particles of the stratified sample.  Stage-isolated: the GPU's own converged
    (H, rho, Omega) of all particles are the inputs of both sides."""
    from parity_util import FLOOR, RTOL_FORCE, ULPS, dev

    ps = _set("C4")
    n = ps.n
    rng = np.random.default_rng(I.SEED_BASE + 78)
    sample = _stratified_sample(ps, np.arange(n, dtype=np.int32), rng)[::16].copy()
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    gd = g.density(ps.h_guess, ps.n_ngb, ps.n_tol)
    assert gd["unconv"] == 0
    H, rho, om = gd["H"], gd["rho"], gd["omega"]
    f32 = torch.float32
    dH, drho, dom, dvel, du_ = dev(H, f32), dev(rho, f32), dev(om, f32), dev(ps.vel, f32), dev(ps.u, f32)
    res = ULPS * 2.0 ** -24
    # R17
    dv = torch.zeros(n, device="cuda"); cv = torch.zeros((n, 3), device="cuda")
    g.sph.sph_velocity_gradients(dvel, dH, drho, dv, cv)
    torch.cuda.synchronize()
    dvn, cvn = dv.cpu().numpy(), cv.cpu().numpy()
    og = O.velocity_gradients(ps.pos, ps.vel, H, rho, kernel=ps.kernel, mass_scalar=ps.mass, active=sample)
    scale = np.abs(ps.vel).max() * 3.0 / H[sample]
    assert np.max(np.abs(dvn[sample] - og["divv"]) / np.maximum(np.abs(og["divv"]), 1e-3 * scale)) < 1e-4
    assert np.max(np.abs(cvn[sample] - og["curlv"]).max(1) / np.maximum(np.abs(og["curlv"]).max(1), 1e-3 * scale)) < 1e-4
    # R18-R20 with the GPU's gradients as the common input
    alpha = np.random.default_rng(5).uniform(0.02, 3.0, n).astype(np.float32)
    kw = dict(alpha_min=0.02, alpha_max=3.0, decay_l=4.0, alpha_cond=0.25, balsara=True)
    acc = torch.zeros((n, 3), device="cuda")
    du, vs, da = (torch.zeros(n, device="cuda") for _ in range(3))
    g.sph.sph_hydro_force_improved(dvel, du_, dH, drho, dom, dev(alpha, f32), dv, cv, acc, du, vs, da, **kw)
    torch.cuda.synchronize()
    of = O.hydro_force_improved(ps.pos, ps.vel, ps.u, H, rho, om, alpha, dvn, cvn, kernel=ps.kernel, mass_scalar=ps.mass, active=sample, **kw)
    ga, gdu = acc.cpu().numpy().astype(np.float64)[sample], du.cpu().numpy().astype(np.float64)[sample]
    tol_a = RTOL_FORCE * np.maximum(np.sqrt((of["acc"] ** 2).sum(1)), FLOOR * of["asum"]) + res * np.sqrt(of["asq"])
    err_a = np.sqrt(((ga - of["acc"]) ** 2).sum(1))
    assert np.all(err_a <= tol_a), float(np.max(err_a / tol_a))
    tol_d = RTOL_FORCE * np.maximum(np.abs(of["dudt"]), FLOOR * of["dusum"]) + res * np.sqrt(of["dusq"])
    err_d = np.abs(gdu - of["dudt"])
    assert np.all(err_d <= tol_d), float(np.max(err_d / tol_d))
    assert np.max(np.abs(vs.cpu().numpy()[sample] - of["vsig"]) / of["vsig"]) < 1e-5
    # R21
    out = torch.zeros(n, device="cuda")
    g.sph.sph_thermal_conduction(du_, dH, drho, out, 0.8, 2.5)
    torch.cuda.synchronize()
    oc = O.thermal_conduction(ps.pos, ps.u, H, rho, kernel=ps.kernel, kappa0=0.8, kappa_exp=2.5, mass_scalar=ps.mass, active=sample)
    tol_c = RTOL_FORCE * np.maximum(np.abs(oc["dudt"]), FLOOR * oc["dusum"]) + res * np.sqrt(oc["dusq"])
    err_c = np.abs(out.cpu().numpy().astype(np.float64)[sample] - oc["dudt"])
    assert np.all(err_c <= tol_c), float(np.max(err_c / tol_c))
    # R23 with the TreePM-like parameters bench.py times (mesh cell = half the mean spacing)
    cell = 0.5 / n ** (1.0 / 3.0)
    gk = dict(G=1.0, r_s=1.25 * cell, r_cut=4.5 * 1.25 * cell, eps=2.0 * cell / 40.0)
    og_ = O.gravity_short(ps.pos, mass_scalar=ps.mass, active=sample, **gk)
    amag = np.sqrt((og_["acc"] ** 2).sum(1))
    g.sph.sph_gravity_short(acc, gk["G"], gk["r_s"], gk["r_cut"], gk["eps"], 0.0, active=dev(sample, torch.int32))
    torch.cuda.synchronize()
    a0 = acc.cpu().numpy().astype(np.float64)[sample]
    err_g = np.sqrt(((a0 - og_["acc"]) ** 2).sum(1))
    tol_g = 1e-4 * np.maximum(amag, 1e-3 * og_["asum"])
    assert np.all(err_g <= tol_g), float(np.max(err_g / tol_g))
    g.sph.sph_gravity_short(acc, gk["G"], gk["r_s"], gk["r_cut"], gk["eps"], 0.5)  # all particles, opening angle 0.5
    torch.cuda.synchronize()
    rel = np.sqrt(((acc.cpu().numpy()[sample] - og_["acc"]) ** 2).sum(1)) / np.maximum(amag, np.median(amag))
    assert np.median(rel) < 5e-3 and np.percentile(rel, 99) < 5e-2, (np.median(rel), np.percentile(rel, 99), rel.max())
    print("C4 full extensions: gradients ok, improved acc/dudt err/tol", float(np.max(err_a / tol_a)), float(np.max(err_d / tol_d)),
          "conduction", float(np.max(err_c / tol_c)), "gravity theta 0", float(np.max(err_g / tol_g)), "theta 0.5 median/99%/max",
          float(np.median(rel)), float(np.percentile(rel, 99)), float(rel.max()))
    g.close()


def test_fullsize_config5_active_subset():
    """configs[4]: the 10^7 set with 1% active by time bin; state = the converged set, actives' h perturbed."""
    ps = _set("C4")
    act = I.config5_active(ps)
    g0 = GpuRun(ps.pos, ps.kernel, ps.mass)
    full = g0.density(ps.h_guess, ps.n_ngb, ps.n_tol)
    g0.close()
    assert full["unconv"] == 0
    hg = I.perturb_h(full["H"], act, I.SEED_BASE + 5)
    ps5 = I.ParticleSet("C5", ps.pos, ps.vel, ps.u, hg, ps.mass, ps.kernel, ps.n_ngb, ps.n_tol, aux=ps.aux)
    g, gd, sample, rep = _sampled_parity(ps5, act, "C5 full e2e")
    H = hg.copy(); H[act] = gd["H"][act]
    rho = full["rho"].copy(); rho[act] = gd["rho"][act]
    om = full["omega"].copy(); om[act] = gd["omega"][act]
    gf = g.force(ps.vel, ps.u, H, rho, om, active=act)
    of = O.hydro_force(ps.pos, ps.vel, ps.u, H, rho, om, kernel=ps.kernel, mass_scalar=ps.mass, active=sample)
    repf = check_force(gf, of, sel=sample, label="C5 full force")
    inact = np.ones(ps.n, bool); inact[act] = False
    assert np.all(gf["acc"][inact] == 7.0)
    print("C5 full", rep, repf, g.sph.stats())
    g.close()
    _cache.clear()
