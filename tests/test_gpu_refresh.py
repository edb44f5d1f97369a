"""sph_refresh_index (index refresh instead of a rebuild for steps with few active particles):
after the particles moved, the refreshed index must give what the oracle gives at the NEW positions -- and what a fresh
build on the GPU gives -- although the octree is still that of the old positions with enlarged cells."""
import numpy as np
import pytest
import torch

from oracle import sph_oracle as O
from paper_2003_10850_b200 import binding as B
from paper_2003_10850_b200 import inputs as I
from parity_util import GpuRun, check_density_e2e, check_force, dev

pytestmark = pytest.mark.gpu


def _moved(ps, frac, seed):
    """Every particle displaced by up to frac * its support-radius guess per axis, wrapped into [0, 1)."""
    rng = np.random.default_rng(seed)
    d = rng.uniform(-1.0, 1.0, (ps.n, 3)) * (frac * ps.h_guess.astype(np.float64))[:, None]
    p = np.mod(ps.pos.astype(np.float64) + d, 1.0).astype(np.float32)
    p[p >= 1.0] = 0.0
    return p


@pytest.mark.parametrize("shape,frac", [("C1", 0.2), ("C2", 0.5), ("C4", 0.3), ("C4", 2.0)])
def test_refreshed_index_against_the_oracle(shape, frac):
    ps = {"C1": lambda: I.config1(12), "C2": lambda: I.config2(20), "C4": lambda: I.config4(24000, 6, m_lo=320, m_hi=8000)}[shape]()
    pos1 = _moved(ps, frac, 11)
    assert np.any(np.abs(pos1 - ps.pos) > 0.5)  # somebody crossed the wall
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    g.density(ps.h_guess, ps.n_ngb, ps.n_tol)  # the index has been used at the old positions
    g.pos.copy_(torch.from_numpy(pos1))
    g.sph.sph_refresh_index(g.pos)
    o = O.density(pos1, ps.h_guess, kernel=ps.kernel, n_target=ps.n_ngb, n_tol=ps.n_tol, mass_scalar=ps.mass)
    gd = g.density(ps.h_guess, ps.n_ngb, ps.n_tol)
    check_density_e2e(gd, o, pos1, ps.h_guess, ps.kernel, ps.mass, ps.n_ngb, ps.n_tol, label=f"{shape} refreshed")
    H, rho, om = (o[k].astype(np.float32) for k in ("H", "rho", "omega"))
    of = O.hydro_force(pos1, ps.vel, ps.u, H, rho, om, kernel=ps.kernel, mass_scalar=ps.mass)
    gf = g.force(ps.vel, ps.u, H, rho, om)
    check_force(gf, of, label=f"{shape} refreshed force")
    # a subset call on the refreshed index
    act = np.sort(np.random.default_rng(3).choice(ps.n, ps.n // 7, replace=False)).astype(np.int32)
    ga = g.density(ps.h_guess, ps.n_ngb, ps.n_tol, active=act)
    assert np.array_equal(ga["Nint"][act], gd["Nint"][act]) and np.allclose(ga["H"][act], gd["H"][act], rtol=1e-6)
    # a fresh build at the new positions: same neighbour sets, hence the same integers; sums in another order
    g2 = GpuRun(pos1, ps.kernel, ps.mass)
    gd2 = g2.density(ps.h_guess, ps.n_ngb, ps.n_tol)
    same = gd["Nint"] == gd2["Nint"]
    assert np.all(same | (o["edge"] != 0))
    assert np.allclose(gd["H"][same], gd2["H"][same], rtol=2e-6) and np.allclose(gd["rho"][same], gd2["rho"][same], rtol=1e-5)
    # refreshing twice, back to the old positions: the cells shrink again (the slack is not cumulative)
    g.pos.copy_(torch.from_numpy(ps.pos))
    g.sph.sph_refresh_index(g.pos)
    g3 = GpuRun(ps.pos, ps.kernel, ps.mass)
    a, b = g.density(ps.h_guess, ps.n_ngb, ps.n_tol), g3.density(ps.h_guess, ps.n_ngb, ps.n_tol)
    assert np.array_equal(a["Nint"], b["Nint"]) and np.array_equal(a["H"], b["H"]) and np.array_equal(a["rho"], b["rho"])
    for x in (g, g2, g3):
        x.close()


def test_gravity_on_a_refreshed_index():
    """The tree walk of sph_gravity_short reads the enlarged cells: the opening criterion only gets more conservative, the
    node moments are recomputed from the new positions."""
    ps = I.config3(8000, 4)
    pos1 = _moved(ps, 0.7, 5)
    kw = dict(G=1.0, r_s=0.03, r_cut=0.135, eps=0.002)
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    g.pos.copy_(torch.from_numpy(pos1))
    g.sph.sph_refresh_index(g.pos)
    o = O.gravity_short(pos1, mass_scalar=ps.mass, **kw)
    amag = np.sqrt((o["acc"] ** 2).sum(1))
    acc = torch.zeros((ps.n, 3), device="cuda")
    g.sph.sph_gravity_short(acc, kw["G"], kw["r_s"], kw["r_cut"], kw["eps"], 0.0)
    a0 = acc.cpu().numpy().astype(np.float64)
    err = np.sqrt(((a0 - o["acc"]) ** 2).sum(1))
    tol = 1e-4 * np.maximum(amag, 1e-3 * o["asum"])
    assert np.all(err <= tol), float(np.max(err / tol))
    g.sph.sph_gravity_short(acc, kw["G"], kw["r_s"], kw["r_cut"], kw["eps"], 0.5)
    rel = np.sqrt(((acc.cpu().numpy() - o["acc"]) ** 2).sum(1)) / np.maximum(amag, np.median(amag))
    assert np.median(rel) < 5e-3 and np.percentile(rel, 99) < 3e-2 and rel.max() < 0.1
    g.close()


def test_refresh_preconditions():
    ps = I.config1(8)
    s = B.Sph(kernel=ps.kernel)
    pos = dev(ps.pos, torch.float32)
    with pytest.raises(B.SphError) as e:
        s.sph_refresh_index(pos)
    assert e.value.code == B.SPH_E_NOINDEX
    s.sph_build_index(pos, None, ps.mass)
    with pytest.raises(B.SphError) as e:
        s.sph_refresh_index(pos[:100].contiguous())
    assert e.value.code == B.SPH_E_ARG
    bad = pos.clone()
    bad[5, 2] = 1.5
    s.sph_refresh_index(bad)  # asynchronous: reported by the next call that looks
    h = dev(ps.h_guess, torch.float32).clone()
    out = [torch.zeros(ps.n, device="cuda") for _ in range(2)] + [torch.zeros(ps.n, device="cuda", dtype=torch.int32)]
    with pytest.raises(B.SphError) as e:
        s.sph_density(h, out[0], out[1], out[2], ps.n_ngb, ps.n_tol)
    assert e.value.code == B.SPH_E_ARG and "position outside" in str(e.value)
    s.sph_build_index(pos, None, ps.mass)
    assert s.sph_density(h, out[0], out[1], out[2], ps.n_ngb, ps.n_tol) == 0
    s.close()
