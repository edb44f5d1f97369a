"""GPU parity of the improved-SPH extension (R17-R20) against the fp64 oracle, through the C
ABI: velocity divergence/curl (sph_velocity_gradients) and the force pass with per-particle alpha, shear limiter and
artificial conduction (sph_hydro_force_improved), on C2- and C4-shaped sets; stage-isolated (a common state feeds both
sides, the oracle's brute-force sums over a sampled active list)."""
import numpy as np
import pytest
import torch

from oracle import sph_oracle as O
from paper_2003_10850_b200 import inputs as I
from parity_util import FLOOR, RTOL_FORCE, ULPS, GpuRun, dev

pytestmark = pytest.mark.gpu


def _state(ps):
    o = O.density(ps.pos, ps.h_guess, kernel=ps.kernel, n_target=ps.n_ngb, n_tol=ps.n_tol, mass_scalar=ps.mass)
    return o["H"].astype(np.float32), o["rho"].astype(np.float32), o["omega"].astype(np.float32)


def _gradients(g, ps, H, rho, active=None):
    n = ps.n
    dv = torch.full((n,), 9.0, device="cuda")
    cv = torch.full((n, 3), 9.0, device="cuda")
    act = None if active is None else dev(active, torch.int32)
    g.sph.sph_velocity_gradients(dev(ps.vel, torch.float32), dev(H, torch.float32), dev(rho, torch.float32), dv, cv, active=act)
    torch.cuda.synchronize()
    return dv.cpu().numpy(), cv.cpu().numpy()


@pytest.mark.parametrize("shape", ["C2", "C4"])
def test_improved_sph_against_the_oracle(shape):
    ps = I.config2(20) if shape == "C2" else I.config4(24000, 6, m_lo=320, m_hi=8000)
    H, rho, om = _state(ps)
    n = ps.n
    rng = np.random.default_rng(5)
    sample = np.sort(rng.choice(n, 1500, replace=False)).astype(np.int32)
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    # R17: all particles on the GPU, the sample by the oracle
    dv, cv = _gradients(g, ps, H, rho)
    og = O.velocity_gradients(ps.pos, ps.vel, H, rho, kernel=ps.kernel, mass_scalar=ps.mass, active=sample)
    # the sums cancel like the force sums do: compare against the magnitude of their terms, ~ |v| / H (R15)
    scale = np.abs(ps.vel).max() * 3.0 / H[sample]
    assert np.max(np.abs(dv[sample] - og["divv"]) / np.maximum(np.abs(og["divv"]), 1e-3 * scale)) < 1e-4
    assert np.max(np.abs(cv[sample] - og["curlv"]).max(1) / np.maximum(np.abs(og["curlv"]).max(1), 1e-3 * scale)) < 1e-4
    # the subset call writes the active entries only, with the same values (other groups, hence another summation order)
    dv2, cv2 = _gradients(g, ps, H, rho, active=sample)
    inact = np.ones(n, bool); inact[sample] = False
    tiny = 1e-5 * np.abs(dv).max()
    assert np.allclose(dv2[sample], dv[sample], rtol=1e-4, atol=tiny) and np.allclose(cv2[sample], cv[sample], rtol=1e-4, atol=tiny)
    assert np.all(dv2[inact] == 9.0) and np.all(cv2[inact] == 9.0)
    # R18-R20: the force pass with the GPU's own gradients as the common input of both sides
    alpha = rng.uniform(0.02, 3.0, n).astype(np.float32)
    kw = dict(alpha_min=0.02, alpha_max=3.0, decay_l=4.0, alpha_cond=0.25, balsara=True)
    of = O.hydro_force_improved(ps.pos, ps.vel, ps.u, H, rho, om, alpha, dv, cv, kernel=ps.kernel, mass_scalar=ps.mass, active=sample, **kw)
    acc = torch.full((n, 3), 7.0, device="cuda")
    du, vs, da = (torch.full((n,), 7.0, device="cuda") for _ in range(3))
    f32 = torch.float32
    g.sph.sph_hydro_force_improved(dev(ps.vel, f32), dev(ps.u, f32), dev(H, f32), dev(rho, f32), dev(om, f32), dev(alpha, f32),
                                   dev(dv, f32), dev(cv, f32), acc, du, vs, da, **kw)
    torch.cuda.synchronize()
    ga, gd, gv, gal = (t.cpu().numpy().astype(np.float64) for t in (acc, du, vs, da))
    res = ULPS * 2.0 ** -24
    tol_a = RTOL_FORCE * np.maximum(np.sqrt((of["acc"] ** 2).sum(1)), FLOOR * of["asum"]) + res * np.sqrt(of["asq"])
    err_a = np.sqrt(((ga[sample] - of["acc"]) ** 2).sum(1))
    assert np.all(err_a <= tol_a), float(np.max(err_a / tol_a))
    tol_d = RTOL_FORCE * np.maximum(np.abs(of["dudt"]), FLOOR * of["dusum"]) + res * np.sqrt(of["dusq"])
    err_d = np.abs(gd[sample] - of["dudt"])
    assert np.all(err_d <= tol_d), float(np.max(err_d / tol_d))
    assert np.max(np.abs(gv[sample] - of["vsig"]) / of["vsig"]) < 1e-5
    assert np.max(np.abs(gal[sample] - of["dalpha"]) / np.maximum(np.abs(of["dalpha"]), 1e-3 * np.abs(of["dalpha"]).max())) < 1e-5
    assert np.abs(of["ducond"]).sum() > 0  # conduction took part
    # reduction on the GPU: constant alpha, limiter and conduction off = the base force pass, bit for bit or nearly
    a0 = np.full(n, 1.0, np.float32)
    g.sph.sph_hydro_force_improved(dev(ps.vel, f32), dev(ps.u, f32), dev(H, f32), dev(rho, f32), dev(om, f32), dev(a0, f32),
                                   dev(dv, f32), dev(cv, f32), acc, du, vs, da, alpha_cond=0.0, balsara=False)
    base = g.force(ps.vel, ps.u, H, rho, om)
    torch.cuda.synchronize()
    assert np.allclose(acc.cpu().numpy(), base["acc"], rtol=2e-5, atol=1e-6 * np.abs(base["acc"]).max())
    assert np.array_equal(vs.cpu().numpy(), base["vsig"])
    print(shape, "improved: acc err/tol", float(np.max(err_a / tol_a)), "dudt err/tol", float(np.max(err_d / tol_d)))
    g.close()


@pytest.mark.parametrize("shape,kexp", [("C2", 2.5), ("C4", 2.5), ("C2", 0.0)])
def test_thermal_conduction_against_the_oracle(shape, kexp):
    """the conduction pair pass on the GPU against the oracle's brute-force sum."""
    ps = I.config2(20) if shape == "C2" else I.config4(24000, 6, m_lo=320, m_hi=8000)
    H, rho, om = _state(ps)
    n = ps.n
    rng = np.random.default_rng(6)
    sample = np.sort(rng.choice(n, 1500, replace=False)).astype(np.int32)
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    f32 = torch.float32
    out = torch.full((n,), 7.0, device="cuda")
    g.sph.sph_thermal_conduction(dev(ps.u, f32), dev(H, f32), dev(rho, f32), out, 0.8, kexp)
    torch.cuda.synchronize()
    o = O.thermal_conduction(ps.pos, ps.u, H, rho, kernel=ps.kernel, kappa0=0.8, kappa_exp=kexp, mass_scalar=ps.mass, active=sample)
    gd = out.cpu().numpy().astype(np.float64)
    tol = RTOL_FORCE * np.maximum(np.abs(o["dudt"]), FLOOR * o["dusum"]) + ULPS * 2.0 ** -24 * np.sqrt(o["dusq"])
    err = np.abs(gd[sample] - o["dudt"])
    assert np.all(err <= tol), float(np.max(err / tol))
    # energy: all particles active, equal masses -> sum du/dt = 0 to rounding
    assert abs(gd.sum()) < 1e-5 * np.abs(gd).sum()
    # active subset: only those entries are written
    out2 = torch.full((n,), 7.0, device="cuda")
    g.sph.sph_thermal_conduction(dev(ps.u, f32), dev(H, f32), dev(rho, f32), out2, 0.8, kexp, active=dev(sample, torch.int32))
    torch.cuda.synchronize()
    o2 = out2.cpu().numpy()
    inact = np.ones(n, bool); inact[sample] = False
    o1 = out.cpu().numpy()
    assert np.allclose(o2[sample], o1[sample], rtol=1e-4, atol=1e-5 * np.abs(o1).max()) and np.all(o2[inact] == 7.0)
    print(shape, kexp, "conduction err/tol", float(np.max(err / tol)))
    g.close()
