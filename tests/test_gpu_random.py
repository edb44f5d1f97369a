"""Randomised GPU parity against the brute-force fp64 oracle: many small seeded sets with random sizes,
boxes, kernels, support radii spread over a decade, clumps, coincident particles and random active
subsets.  Stage-isolated protocol (one evaluation at given H; force with given state), so every case is
an exact definition on both sides.  Aims at the index/walk/gather edge cases: ragged chunks, groups at
box faces and corners (all three frame modes), single-particle leaves, oversize leaves."""
import numpy as np
import pytest

from oracle import sph_oracle as O
from parity_util import GpuRun, check_density_stage, check_force

pytestmark = pytest.mark.gpu


def _random_set(rng):
    n = int(rng.choice([1, 2, 3, 17, 33, 100, 257, 700, 1500, 3000]))
    box = float(rng.choice([1.0, 0.37, 2.5]))
    kind = rng.integers(0, 3)
    if kind == 0:  # uniform
        pos = rng.uniform(0, 1, (n, 3))
    elif kind == 1:  # a few tight clumps + background, some exactly coincident particles
        c = rng.uniform(0, 1, (max(1, n // 200 + 1), 3))
        pos = c[rng.integers(0, len(c), n)] + rng.normal(0, 10.0 ** rng.uniform(-3, -1.3), (n, 3))
        k = n // 10
        if k:
            pos[rng.integers(0, n, k)] = pos[rng.integers(0, n, k)]
    else:  # hugging the faces and corners of the box
        pos = rng.uniform(0, 1, (n, 3))
        m = rng.random((n, 3)) < 0.5
        pos[m] = np.where(rng.random(m.sum()) < 0.5, 1e-3, 1 - 1e-3) * rng.uniform(0.0, 1.0, m.sum()) + \
            np.where(rng.random(m.sum()) < 0.5, 0.0, 0.999)
    pos = (pos % 1.0) * box
    pos32 = pos.astype(np.float32)
    pos32[pos32 >= np.float32(box)] = 0.0
    # support radii: log-uniform over up to a decade above the mean spacing, capped below box / 2
    d = box / max(n, 2) ** (1.0 / 3.0)
    # (not below ~1.3 spacings: a support holding only one or two far neighbours sums nothing but kernel
    # tails (1 - q)^7, whose fp32 relative error 7 eps / (1 - q) exceeds any fixed relative tolerance)
    lo, hi = d * 10.0 ** rng.uniform(0.1, 0.4), d * 10.0 ** rng.uniform(0.4, 1.0)
    h = np.minimum(np.exp(rng.uniform(np.log(lo), np.log(hi), n)), 0.45 * box).astype(np.float32)
    vel = rng.normal(0, 0.3, (n, 3)).astype(np.float32)
    u = np.exp(rng.uniform(np.log(0.5), np.log(2.0), n)).astype(np.float32)
    return n, box, pos32, h, vel, u


@pytest.mark.parametrize("seed", range(24))
def test_random_small_sets_against_bruteforce(seed):
    rng = np.random.default_rng(7_2003_10850 + seed)
    n, box, pos, h, vel, u = _random_set(rng)
    kernel = int(rng.integers(0, 2))
    mass = 1.0 / n
    use_mass = bool(rng.integers(0, 2))
    marr = np.exp(rng.uniform(-1, 1, n)).astype(np.float32) * np.float32(mass) if use_mass else None
    active = None
    if n > 3 and rng.random() < 0.5:
        active = np.sort(rng.choice(n, int(rng.integers(1, n)), replace=False)).astype(np.int32)
    gcap = int(rng.choice([0, 1, 3, 8, 16, 32]))
    g = GpuRun(pos, kernel, mass, box=box, mass=marr, group_cap=gcap, group_node=int(rng.choice([0, 32, 64])))
    label = f"seed {seed} n {n} box {box} k {kernel} mass {use_mass} act {None if active is None else len(active)} cap {gcap}"
    oe = O.density_eval(pos, h, kernel=kernel, mass_scalar=mass, mass=marr, box=box, active=active, brute=True)
    ge = g.density(h, 50.0, float("inf"), active=active)
    assert ge["unconv"] == 0
    check_density_stage(ge, oe, sel=active, label=label)
    # force with the oracle's densities (all particles) as the common state
    of_all = O.density_eval(pos, h, kernel=kernel, mass_scalar=mass, mass=marr, box=box, brute=True)
    rho = of_all["rho"].astype(np.float32)
    om = of_all["omega"].astype(np.float32)
    # particles (nearly) alone in their support have Omega = 0 up to rounding; A = P / (Omega rho^2) then
    # multiplies kernel tails that vanish: an ill-conditioned input, not a regime of the method.  Any
    # finite value is an equally arbitrary common input for both sides.
    om[np.abs(om) < 1e-3] = 1.0
    of = O.hydro_force(pos, vel, u, h, rho, om, kernel=kernel, mass_scalar=mass, mass=marr, box=box, active=active,
                       brute=True)
    gf = g.force(vel, u, h, rho, om, active=active)
    check_force(gf, of, sel=active, label=label)
    if active is not None:
        inact = np.ones(n, bool)
        inact[active] = False
        assert np.all(ge["rho"][inact] == -1) and np.all(gf["dudt"][inact] == 7.0)
    g.close()
