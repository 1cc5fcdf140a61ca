"""gfmc_moments_static -- the entry point for callers that cannot allocate device memory (`-m gpu`).

Some users of libgfmc.so may not call cudaMalloc when they need moments: their process handed the whole GPU to its own pool
allocator, or an allocation call would break a stream capture running in another thread, or would stall a latency-critical loop.
For them the library keeps the scratch of the shared-memory-resident moments path in a fixed array inside its own image
(include/gfmc.h).  That array is shared by all calls and keeps the previous call's contents, so what has to be shown is that a call
gives the existing path's answer (a) on first use in a fresh process and (b) right after another call with different sizes left
its data behind.  Both are checked against gfmc_create + gfmc_moments within the moment tolerance of the other GPU tests (1e-10; the
two paths launch the same kernels, so the difference is in fact zero).

This file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here cannot hide the parity tests."""
import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl

pytestmark = pytest.mark.gpu

MU_TOL = 1e-10          # tests/test_gpu_parity.py


def _existing_path(L, M, JH, S, sites):
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=0.05, max_batch_sites=len(sites))
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments(ctx, sites)
    assert g.gfmc_launch_counts(ctx)[0] == 1          # the resident kernel: one launch for all M/2 steps
    g.gfmc_destroy(ctx)
    return mu


def _static_path(L, M, JH, S, sites, out=None):
    import torch
    mu = g.gfmc_moments_static(L, M, 1.0, JH, torch.from_numpy(S).cuda(), torch.from_numpy(sites).cuda(), out=out)
    return mu.cpu().numpy()


def test_two_calls_in_a_row_match_the_existing_path():
    """Call 1 fills much of the shared scratch array (L = 8, M = 128, 300 sites); call 2 is smaller in every dimension (L = 6:
    another slot packing, M = 32, 50 sites, other spins and coupling) and must not see what call 1 left behind; call 3 repeats call
    1's shape at L = 10 (several sites per thread) into a caller-provided output."""
    import torch
    cases = [(8, 128, 4.0, 300), (6, 32, 2.5, 50), (10, 24, 4.0, 150)]
    for k, (L, M, JH, n) in enumerate(cases):
        S = wl.make_spins(L, seed=900 + k)
        sites = np.random.default_rng(40 + k).choice(L ** 3, size=n, replace=False).astype(np.int32)
        out = torch.full((n, M, 2, 2), float("nan"), dtype=torch.complex128, device="cuda") if k == 2 else None
        got = _static_path(L, M, JH, S, sites, out=out)
        ref = _existing_path(L, M, JH, S, sites)
        assert np.isfinite(got.view(np.float64)).all()
        assert np.abs(got - ref).max() <= MU_TOL, (L, M, n)
        assert np.abs(got[:, 0] - np.eye(2)).max() == 0.0          # mu_0 = identity (Eq. (25) at n = 0)


def test_same_call_twice_is_bitwise_repeatable():
    L, M, n = 8, 64, 512
    S = wl.make_spins(L, seed=77)
    sites = np.arange(n, dtype=np.int32)
    a = _static_path(L, M, 4.0, S, sites)
    b = _static_path(L, M, 4.0, S, sites)
    assert np.array_equal(a.view(np.float64), b.view(np.float64))


def test_sizes_beyond_the_fixed_scratch_are_refused():
    import torch
    S = torch.from_numpy(wl.make_spins(8, seed=1)).cuda()
    n = 2 * g.GFMC_STATIC_MAX_STEP_SITES // 256 + 1               # (M/2) * n just above the maximum at M = 256
    sites = torch.zeros(n, dtype=torch.int32, device="cuda")
    with pytest.raises(g.GfmcError, match="exceeds the fixed scratch array's maximum") as ei:
        g.gfmc_moments_static(8, 256, 1.0, 4.0, S, sites)
    assert ei.value.code == -1
    g.gfmc_moments_static(8, 256, 1.0, 4.0, S, sites[:n - 1])     # exactly at the maximum: accepted
    S16 = torch.from_numpy(wl.make_spins(16, seed=1)).cuda()
    with pytest.raises(g.GfmcError, match="outside 2..12"):
        g.gfmc_moments_static(16, 8, 1.0, 4.0, S16, sites[:4])
    with pytest.raises(g.GfmcError, match="even"):
        g.gfmc_moments_static(8, 7, 1.0, 4.0, S, sites[:4])
    empty = g.gfmc_moments_static(8, 8, 1.0, 4.0, S, sites[:0])
    assert tuple(empty.shape) == (0, 8, 2, 2)
