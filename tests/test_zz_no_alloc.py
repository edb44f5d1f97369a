"""sph_compact_flags_noalloc: the stream compaction of the active-list step with its scratch in a fixed file-scope
device array (no cudaMalloc / cudaFree: for callers under CUDA graph capture, serving loops, harnesses that forbid
allocation) against the existing path, sph_compact_flags (context scratch, grows by cudaMalloc) -- integer work, so
the comparison is bit-exact.  Collected last on purpose (the file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2003_10850_b200 import binding as B

pytestmark = pytest.mark.gpu


def _flags(n, frac, seed):
    rng = np.random.default_rng(seed)
    return (rng.random(n) < frac).astype(np.uint32)


def _call(sph, f_np, noalloc, fill):
    n = len(f_np)
    flags = torch.from_numpy(f_np).cuda()
    ids = torch.full((n,), fill, device="cuda", dtype=torch.int32)
    cnt = torch.from_numpy(np.array([0xFFFFFFFF], np.uint32)).cuda()
    sph.sph_compact_flags(flags, ids, cnt, noalloc=noalloc)
    torch.cuda.synchronize()
    return ids.cpu().numpy(), int(cnt.cpu().numpy()[0])


def test_noalloc_compaction_matches_the_existing_path_on_two_calls_in_a_row():
    sph = B.Sph()
    # two calls in a row on the shared scratch: a large one (733 blocks of 4096 flags, ragged tail), then a smaller one
    # with other flags -- whatever the first call left in the array must not reach the second
    cases = [(3_000_001, 0.37, 1), (70_001, 0.02, 2), (4096, 1.0, 3), (1, 1.0, 4), (5000, 0.0, 5)]
    for n, frac, seed in cases:
        f = _flags(n, frac, seed)
        want = np.flatnonzero(f).astype(np.int32)
        ids0, c0 = _call(sph, f, False, -7)
        ids1, c1 = _call(sph, f, True, -7)
        assert c0 == c1 == len(want), (n, c0, c1, len(want))
        assert np.array_equal(ids1, ids0)                                    # bit-exact against the existing path ...
        assert np.array_equal(ids1[:c1], want) and np.all(ids1[c1:] == -7)   # ... which is the plain definition
    # the same inputs again, in the other order of sizes: same answers (nothing of an earlier call is read)
    for n, frac, seed in reversed(cases):
        f = _flags(n, frac, seed)
        ids1, c1 = _call(sph, f, True, -3)
        assert c1 == int(f.sum()) and np.array_equal(ids1[:c1], np.flatnonzero(f).astype(np.int32))
    sph.close()


def test_noalloc_compaction_allocates_nothing_and_rejects_oversize():
    sph = B.Sph()
    n = 1_000_000
    f = torch.from_numpy(_flags(n, 0.5, 9)).cuda()
    ids = torch.zeros(n, device="cuda", dtype=torch.int32)
    cnt = torch.zeros(1, device="cuda", dtype=torch.int32).view(torch.uint32)
    sph.sph_compact_flags(f, ids, cnt, noalloc=True)  # (first call on the device: asks for the scratch array's address)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        sph.sph_compact_flags(f, ids, cnt, noalloc=True)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0  # the device's free memory did not move
    assert int(cnt.cpu().numpy()[0]) == int(f.cpu().numpy().sum())
    # beyond the fixed scratch: a clear error, nothing launched (the arrays are not touched: sizes are not looked at)
    lib = B.load()
    rc = lib.sph_compact_flags_noalloc(sph._h, C.c_int64(B.COMPACT_NOALLOC_MAX + 1), C.c_void_p(f.data_ptr()), C.c_void_p(ids.data_ptr()),
                                       C.c_void_p(cnt.data_ptr()))
    assert rc == B.SPH_E_ARG
    msg = lib.sph_last_error(sph._h).decode()
    assert "SPH_COMPACT_NOALLOC_MAX" in msg and str(B.COMPACT_NOALLOC_MAX) in msg
    # the limit itself is accepted by the argument check of the allocating path's twin (not run: 256 MB of flags)
    assert lib.sph_compact_flags_noalloc(sph._h, C.c_int64(-1), None, None, C.c_void_p(cnt.data_ptr())) == B.SPH_E_ARG
    # empty input: count = 0
    e = torch.zeros(0, device="cuda", dtype=torch.int32)
    sph.sph_compact_flags(e.view(torch.uint32), e, cnt, noalloc=True)
    torch.cuda.synchronize()
    assert int(cnt.cpu().numpy()[0]) == 0
    sph.close()


def test_noalloc_compaction_under_cuda_graph_capture():
    """The use case: the call is captured into a CUDA graph (stream capture forbids cudaMalloc / cudaFree) and replayed on
    new flags; the allocating path is not captured.  The first call on the device is made before the capture."""
    s = torch.cuda.Stream()
    sph = B.Sph(stream=s)
    n = 300_000
    f_np = _flags(n, 0.3, 21)
    flags = torch.from_numpy(f_np).cuda()
    ids = torch.full((n,), -1, device="cuda", dtype=torch.int32)
    cnt = torch.zeros(1, device="cuda", dtype=torch.int32).view(torch.uint32)
    with torch.cuda.stream(s):
        sph.sph_compact_flags(flags, ids, cnt, noalloc=True)  # set-up call, not captured
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        sph.sph_compact_flags(flags, ids, cnt, noalloc=True)
    for seed in (22, 23):
        f_np = _flags(n, 0.1 * (seed - 20), seed)
        flags.copy_(torch.from_numpy(f_np).cuda())
        ids.fill_(-1)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        want = np.flatnonzero(f_np).astype(np.int32)
        c = int(cnt.cpu().numpy()[0])
        assert c == len(want) and np.array_equal(ids.cpu().numpy()[:c], want)
    del g
    sph.close()
