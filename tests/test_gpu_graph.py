"""sph_build_index replays its launch sequence from a CUDA graph from the third identical call on (same n and the same
device arrays, a stream other than the legacy default one): the replayed index must be the one a fresh context builds
from the arrays' CURRENT contents."""
import numpy as np
import pytest
import torch

from paper_2003_10850_b200 import binding as B
from paper_2003_10850_b200 import inputs as I
from parity_util import dev

pytestmark = pytest.mark.gpu


def _density(sph, ps, n):
    h = dev(ps.h_guess, torch.float32).clone()
    rho, om = torch.zeros(n, device="cuda"), torch.zeros(n, device="cuda")
    ngb = torch.zeros(n, device="cuda", dtype=torch.int32)
    assert sph.sph_density(h, rho, om, ngb, ps.n_ngb, ps.n_tol) == 0
    torch.cuda.synchronize()
    return h.cpu().numpy(), rho.cpu().numpy(), ngb.cpu().numpy()


@pytest.mark.parametrize("shape", ["C1", "C3"])
def test_index_build_graph_replay(shape):
    ps = I.config1(10) if shape == "C1" else I.config3(20000, 3)
    n = ps.n
    rng = np.random.default_rng(4)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        sph = B.Sph(kernel=ps.kernel, stream=side)
        pos = dev(ps.pos, torch.float32)
        launches = []
        for k in range(5):
            # new positions in the SAME device array before every build (a shuffle + a shift through the wall)
            p_np = np.mod(ps.pos[rng.permutation(n)].astype(np.float64) + 0.137 * k, 1.0).astype(np.float32)
            p_np[p_np >= 1.0] = 0.0
            pos.copy_(torch.from_numpy(p_np))
            l0 = sph.stats()["launches"]
            sph.sph_build_index(pos, None, ps.mass)   # k = 0 direct, k = 1 captures, k >= 2 replay
            got = _density(sph, ps, n)
            launches.append(sph.stats()["launches"] - l0)
            with torch.cuda.stream(torch.cuda.default_stream()):
                ref = B.Sph(kernel=ps.kernel)
                ref.sph_build_index(dev(p_np, torch.float32), None, ps.mass)
                want = _density(ref, ps, n)
                ref.close()
            for a, b in zip(got, want):
                assert np.array_equal(a, b), (shape, k)
        assert len(set(launches)) == 1  # the launch counter counts the replayed kernels as well
        # another array: direct launches again, same results
        pos2 = pos.clone()
        sph.sph_build_index(pos2, None, ps.mass)
        for a, b in zip(_density(sph, ps, n), got):
            assert np.array_equal(a, b)
        sph.close()
    side.synchronize()
