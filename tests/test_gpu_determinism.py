"""Race stress of the streaming kernel's synchronisation protocols (`-m gpu`) -- the stand-in for compute-sanitizer's racecheck,
which is closed on this pool (profiles/r2_sanitizer.md).

Every reduction of the fused step has a fixed order, so its results are bit-reproducible BY DESIGN; the rings' depths change when a
stage is refilled relative to when it is read, but never what is computed.  A missing or misplaced synchronisation (a stage read
before its bulk copy landed, refilled while a warp still reads it, an in-place overwrite of r_{m-2} seen by another thread) therefore
shows up as a bitwise difference between repetitions or between ring depths.  All three modes, the balanced work list (L = 16), the
run-time-L kernel with its CTA-wide R_prev ring (L = 20) and the y-tiled compile-time kernel (L = 32)."""
import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl

pytestmark = pytest.mark.gpu

DEPTHS = [(0, 0), (3, 1), (3, 2), (4, 1), (4, 2), (5, 1), (6, 1)]


@pytest.mark.parametrize("mode", ["hund", "ph", "dex"])
@pytest.mark.parametrize("L,M,n", [(16, 48, 512), (20, 24, 150), (32, 32, 320)])
def test_moments_are_bitwise_identical_across_repetitions_and_ring_depths(oracle, mode, L, M, n):
    S = wl.make_spins(L, seed=400 + L)
    sites = np.random.default_rng(L).choice(L ** 3, size=n, replace=False).astype(np.int32)
    prop = wl.make_spins(L, seed=401 + L)[sites]
    kw = dict(hund={}, ph=dict(ph_symmetry=1), dex=dict(model=g.GFMC_MODEL_DEX_INF))[mode]
    first, used = None, 0
    for nc, np_ in DEPTHS:
        try:
            ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=8.0, T=0.05, max_batch_sites=n, ring_stages_cur=nc, ring_stages_prev=np_, **kw)
        except g.GfmcError:
            continue                                   # this depth does not fit shared memory for this lattice / mode
        g.gfmc_set_spins(ctx, S)
        for rep in range(4):
            mu = g.gfmc_moments_ov(ctx, sites, prop) if mode == "dex" else g.gfmc_moments(ctx, sites)
            if first is None:
                first = mu
            assert np.array_equal(mu, first), (nc, np_, rep, np.abs(mu - first).max())
        g.gfmc_destroy(ctx)
        used += 1
    assert used >= 4
    sub = np.arange(0, n, max(1, n // 6))
    if mode == "dex":
        ref = oracle.dex_moments_many(L, 1.0, S, sites[sub], prop[sub], M, nthreads=8)
        scale = np.maximum(1.0, np.abs(ref[:, 0, 1, 1].real))[:, None, None, None]
    else:
        ref = oracle.moments_many(L, 1.0, 8.0, S, sites[sub], M, nthreads=8)
        scale = 1.0
    assert (np.abs(first[sub] - ref) / scale).max() <= 1e-10


def test_sanitizer_cases_run_clean():
    """The invocations kept for compute-sanitizer (tests/sanitizer_cases.py) at least run to completion as a plain GPU test."""
    from tests.sanitizer_cases import sanitizer_cases
    sanitizer_cases()
