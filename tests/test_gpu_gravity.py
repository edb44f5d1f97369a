"""GPU parity of the short-range Barnes-Hut gravity (sph_gravity_short; R23) against the oracle's
direct summation: exact (to fp32 pair arithmetic) for an opening angle of zero, within the multipole error of the
opening criterion otherwise."""
import numpy as np
import pytest
import torch

from oracle import sph_oracle as O
from paper_2003_10850_b200 import inputs as I
from parity_util import GpuRun, dev

pytestmark = pytest.mark.gpu


def _run(g, n, theta, active=None, **kw):
    acc = torch.full((n, 3), 7.0, device="cuda")
    g.sph.sph_gravity_short(acc, kw["G"], kw["r_s"], kw["r_cut"], kw["eps"], theta, active=None if active is None else dev(active, torch.int32))
    torch.cuda.synchronize()
    return acc.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("shape", ["C1", "C3"])
def test_gravity_against_direct_summation(shape):
    ps = I.config1(14) if shape == "C1" else I.config3(8000, 4)
    n = ps.n
    kw = dict(G=1.0, r_s=0.03, r_cut=0.135, eps=0.002)
    o = O.gravity_short(ps.pos, mass_scalar=ps.mass, **kw)
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    amag = np.sqrt((o["acc"] ** 2).sum(1))
    # theta = 0: every cell is opened, the pair set is the oracle's
    a0 = _run(g, n, 0.0, **kw)
    err = np.sqrt(((a0 - o["acc"]) ** 2).sum(1))
    tol = 1e-4 * np.maximum(amag, 1e-3 * o["asum"])
    assert np.all(err <= tol), float(np.max(err / tol))
    assert np.all(np.abs(a0.sum(0)) < 1e-5 * np.abs(a0).sum(0))  # momentum
    # theta = 0.5: monopole approximation; errors relative to the typical force of the set
    a5 = _run(g, n, 0.5, **kw)
    rel = np.sqrt(((a5 - o["acc"]) ** 2).sum(1)) / np.maximum(amag, np.median(amag))
    assert np.median(rel) < 5e-3 and np.percentile(rel, 99) < 3e-2 and rel.max() < 0.1, (np.median(rel), np.percentile(rel, 99), rel.max())
    if shape == "C3":
        assert np.percentile(rel, 90) > 1e-6  # (cells really were accepted; in the uniform C1 set no cell inside r_cut is small enough)
    a2 = _run(g, n, 0.25, **kw)
    rel2 = np.sqrt(((a2 - o["acc"]) ** 2).sum(1)) / np.maximum(amag, np.median(amag))
    assert np.mean(rel2) <= np.mean(rel)  # a smaller opening angle is at least as accurate
    # active subset: only those entries are written, same values as the all-active call
    rng = np.random.default_rng(3)
    act = np.sort(rng.choice(n, 700, replace=False)).astype(np.int32)
    asub = _run(g, n, 0.0, active=act, **kw)
    inact = np.ones(n, bool); inact[act] = False
    assert np.all(asub[inact] == 7.0) and np.allclose(asub[act], a0[act], rtol=1e-4, atol=1e-6 * amag.max())
    print(shape, "gravity: theta 0 err/tol", float(np.max(err / tol)), "theta 0.5 median/99%/max rel err", np.median(rel), np.percentile(rel, 99), rel.max())
    g.close()


def test_gravity_with_particle_masses():
    """Per-particle masses (a factor 30 between the lightest and the heaviest): the node moments weight the centres of mass,
    the direct sum of the oracle weights every pair term."""
    ps = I.config3(6000, 3)
    n = ps.n
    rng = np.random.default_rng(12)
    m = (ps.mass * np.exp(rng.uniform(-1.7, 1.7, n))).astype(np.float32)
    kw = dict(G=1.0, r_s=0.03, r_cut=0.135, eps=0.002)
    o = O.gravity_short(ps.pos, mass=m, **kw)
    g = GpuRun(ps.pos, ps.kernel, 1.0, mass=m)
    amag = np.sqrt((o["acc"] ** 2).sum(1))
    a0 = _run(g, n, 0.0, **kw)
    err = np.sqrt(((a0 - o["acc"]) ** 2).sum(1))
    tol = 1e-4 * np.maximum(amag, 1e-3 * o["asum"])
    assert np.all(err <= tol), float(np.max(err / tol))
    mom = (m[:, None].astype(np.float64) * a0).sum(0)  # total momentum change: pair terms m_i m_j antisymmetric
    assert np.all(np.abs(mom) < 1e-5 * (m[:, None] * np.abs(a0)).sum(0))
    a5 = _run(g, n, 0.5, **kw)
    rel = np.sqrt(((a5 - o["acc"]) ** 2).sum(1)) / np.maximum(amag, np.median(amag))
    assert np.median(rel) < 5e-3 and np.percentile(rel, 99) < 3e-2 and rel.max() < 0.15, (np.median(rel), np.percentile(rel, 99), rel.max())
    g.close()


def test_gravity_argument_checks():
    from paper_2003_10850_b200 import binding as B

    ps = I.config1(8)
    g = GpuRun(ps.pos, ps.kernel, ps.mass)
    acc = torch.zeros((ps.n, 3), device="cuda")
    with pytest.raises(B.SphError) as e:
        g.sph.sph_gravity_short(acc, 1.0, 0.05, 0.6, 0.0, 0.5)  # r_cut >= box / 2
    assert e.value.code == B.SPH_E_ARG
    g.close()
