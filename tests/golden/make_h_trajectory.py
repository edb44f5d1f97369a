"""Writes tests/golden/h_trajectory.txt: the h-iteration trajectories (rule R7 of DESIGN.md) of a seeded clustered
set, computed by the fp64 oracle ALONE (this script imports nothing of the CUDA path but the arithmetic-free input
generator).  The file freezes the rule: the paper fixes nothing about it ("multiple iterations", §1), so a
change of oracle/sph_oracle.c that moves any of these numbers must come with a new pin and a DESIGN.md reading.

    python tests/golden/make_h_trajectory.py        # rewrites the file
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
from oracle import sph_oracle as O  # noqa: E402
from paper_2003_10850_b200 import inputs as I  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "h_trajectory.txt")


def trajectories():
    """(particle id, evaluations, flags, H after 1, 2, 3 evaluations, final H) of 96 particles of a small C3-like set
    (guesses spread by e^+-0.5 so that clamps and brackets occur), both count modes."""
    ps = I.config3(4096, 4)
    rng = np.random.default_rng(I.SEED_BASE + 31)
    h = (ps.h_guess.astype(np.float64) * np.exp(rng.uniform(-0.5, 0.5, ps.n))).astype(np.float32)
    ids = np.sort(rng.choice(ps.n, 48, replace=False)).astype(np.int32)
    rows = []
    for mode in (0, 1):
        kw = dict(kernel=ps.kernel, n_target=ps.n_ngb, n_tol=ps.n_tol, mass_scalar=ps.mass, active=ids, count_mode=mode)
        part = [O.density(ps.pos, h, max_iter=k, **kw)["H"] for k in (1, 2, 3)]
        full = O.density(ps.pos, h, **kw)
        for j, i in enumerate(ids):
            rows.append((int(i) + mode * ps.n, int(full["iters"][j]), int(full["flags"][j]),
                         float(part[0][j]), float(part[1][j]), float(part[2][j]), float(full["H"][j])))
    return rows


if __name__ == "__main__":
    with open(OUT, "w") as f:
        f.write("# h-iteration trajectories of the fp64 oracle (rule R7, DESIGN.md); written by make_h_trajectory.py\n")
        f.write("# id(+n for count_mode 1)  evaluations  flags  H_after_1  H_after_2  H_after_3  H_final   (C99 hex floats)\n")
        for r in trajectories():
            f.write("%d %d %d %s %s %s %s\n" % (r[0], r[1], r[2], *[x.hex() for x in r[3:]]))
    print("wrote", OUT)
