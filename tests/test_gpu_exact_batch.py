"""GPU parity of GFMC_BATCH_EXACT (exactness inside a batch) against oracle/gfmc_oracle_exact.c (`-m gpu`).

The CUDA path applies the Dyson identity as one rank-2 Woodbury update of all later Green blocks per accepted site; the oracle
solves the full 2|U| x 2|U| system per site and energy.  Same algebra, different arithmetic, same inputs: Delta S within
1e-9 * max(1, |Delta S|), decisions identical away from ties, spins bit-identical."""
import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl

pytestmark = pytest.mark.gpu

DS_RTOL = 1e-9
TIE = 1e-8


def _ds_close(a, b):
    return np.abs(a - b) <= DS_RTOL * np.maximum(1.0, np.abs(b))


@pytest.mark.parametrize("L,M,K,n,kernel,T", [
    (4, 32, 64, 8, 0, 0.05),      # small lattice: the streaming kernel is forced (the read-out needs the vectors in global memory)
    (4, 64, 128, 16, 1, 0.2),     # Lorentz kernel (the paper's), half of a colour class in one batch
    (6, 48, 100, 12, 0, 0.05),    # K not a power of two: direct-sum reconstruction of the P^2 blocks
    (8, 64, 128, 24, 1, 0.05),
    (16, 32, 64, 32, 0, 0.02),    # config 3's lattice
    (20, 16, 32, 10, 0, 0.05),    # run-time-L streaming kernel
    (32, 16, 32, 6, 0, 0.02),     # config 4's lattice, y-tiled work items
])
def test_exact_update_batch_matches_oracle(oracle, L, M, K, n, kernel, T):
    JH = 8.0 if L >= 16 else 4.0
    S = wl.make_spins(L, seed=200 + L)
    rng = np.random.default_rng(L * 7 + n)
    sites = np.sort(rng.choice(wl.colour_sites(L, 0), size=n, replace=False)).astype(np.int32)
    if L <= 8:
        sites[1] = sites[0] + 2                 # second neighbours along x: the largest inter-site Green's function of one colour
        sites = np.unique(sites).astype(np.int32); n = len(sites)
    prop = wl.make_spins(L, seed=201 + L)[sites]
    uni = 1.0 - rng.random(n)
    uni[: n // 2 : 2] = 1e-300                        # make sure several early trials are accepted: the later ones must see them
    ref_dS, ref_acc = oracle.exact_batch_dS(L, 1.0, JH, T, 0.0, M, K, kernel, 4.0, S, sites, prop, uni, nthreads=8)
    frozen = np.array([oracle.site_dS(L, 1.0, JH, T, 0.0, M, K, kernel, 4.0, S, int(s), prop[j]) for j, s in enumerate(sites)])
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=T, n_energy=K, kernel=kernel, max_batch_sites=max(n, 64), exact_batch_sites=n)
    g.gfmc_set_spins(ctx, S)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_EXACT)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop, uni)
    assert g.gfmc_launch_counts(ctx)[0] == M - 1                           # plain recursion: M-1 fused steps, no doubling
    S_gpu = g.gfmc_get_spins(ctx)
    margin = -ref_dS - np.log(uni)
    assert (np.abs(margin) > TIE).all(), "a decision fell inside the tie window; pick another seed"
    assert np.array_equal(acc, ref_acc)
    assert _ds_close(dS, ref_dS).all(), np.abs(dS - ref_dS).max()
    S_ref = S.copy(); S_ref[sites[ref_acc == 1]] = prop[ref_acc == 1]
    assert np.array_equal(S_gpu, S_ref)
    assert ref_acc[: n // 2].sum() >= 2 and dS[0] == pytest.approx(frozen[0], rel=1e-9, abs=1e-9)    # the first site has nothing to see
    if L <= 8:       # (on large lattices a short recursion never connects far-apart sites: their cross moments are exactly zero)
        assert np.abs(ref_dS - frozen).max() > 1e-6                        # ... and the correction is not a no-op on this input
    # the same context in the default mode is the frozen batch again
    g.gfmc_set_spins(ctx, S)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_FROZEN)
    dS_f, _ = g.gfmc_update_batch(ctx, sites, prop, uni)
    assert _ds_close(dS_f, frozen).all()
    g.gfmc_destroy(ctx)


@pytest.mark.parametrize("L,M,K,kernel", [(16, 24, 48, 0), (32, 16, 32, 1)])
def test_exact_update_batch_near_neighbours_on_large_lattices(oracle, L, M, K, kernel):
    """Large lattices with a CLUSTER of same-colour near neighbours in one batch (second neighbours along x, y and z, diagonal
    neighbours, across the periodic wrap in z and across the y-tile boundary of the L = 32 work items): the cross moments between
    them are non-zero from the second step on, so a wrong cross block -- in particular cross_readout_kernel's y-tiled addressing --
    changes Delta S.  (The random far-apart sites of the test above have exactly zero cross moments at these M.)"""
    JH, T = 8.0, 0.05
    S = wl.make_spins(L, seed=400 + L)
    idx = lambda x, y, z: (x % L) + L * ((y % L) + L * (z % L))
    x0, y0, z0 = 5, L // 2 - 1, L - 1                     # y0 + 2 crosses the middle of the lattice (tile edge at L = 32), z0 + 2 wraps
    sites = np.array([idx(x0, y0, z0), idx(x0 + 2, y0, z0), idx(x0, y0 + 2, z0), idx(x0, y0, z0 + 2), idx(x0 + 1, y0 + 1, z0),
                      idx(x0 + 1, y0, z0 + 1), idx(x0, y0 - 1, z0 - 1), idx(x0 - 2, y0, z0), idx(x0 + 9, y0 + 5, z0 + 8)], dtype=np.int32)
    assert len(set(sites.tolist())) == len(sites) and len({(s % L + (s // L) % L + s // (L * L)) % 2 for s in sites.tolist()}) == 1
    n = len(sites)
    prop = wl.make_spins(L, seed=401 + L)[sites]
    uni = 1.0 - np.random.default_rng(L).random(n)
    uni[:6] = 1e-300                                      # the cluster's first six trials are accepted; the later ones must see them
    ref_dS, ref_acc = oracle.exact_batch_dS(L, 1.0, JH, T, 0.0, M, K, kernel, 4.0, S, sites, prop, uni, nthreads=8)
    frozen = np.array([oracle.site_dS(L, 1.0, JH, T, 0.0, M, K, kernel, 4.0, S, int(s), prop[j]) for j, s in enumerate(sites)])
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=T, n_energy=K, kernel=kernel, max_batch_sites=64, exact_batch_sites=n)
    g.gfmc_set_spins(ctx, S)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_EXACT)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop, uni)
    S_gpu = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    margin = -ref_dS - np.log(uni)
    assert (np.abs(margin) > TIE).all(), "a decision fell inside the tie window; pick another seed"
    assert np.array_equal(acc, ref_acc) and ref_acc[:6].all()
    assert _ds_close(dS, ref_dS).all(), np.abs(dS - ref_dS).max()
    S_ref = S.copy(); S_ref[sites[ref_acc == 1]] = prop[ref_acc == 1]
    assert np.array_equal(S_gpu, S_ref)
    assert np.abs(ref_dS[1:8] - frozen[1:8]).min() > 1e-7     # every later site of the cluster feels the earlier flips ...
    assert abs(ref_dS[8] - frozen[8]) < 1e-12                 # ... and the far-away one does not


@pytest.mark.parametrize("L,M,K,B,ns,kernel", [(4, 32, 64, 8, 2, 1), (4, 24, 48, 1, 1, 0), (16, 12, 24, 16, 1, 0)])
def test_exact_sweep_matches_oracle(oracle, L, M, K, B, ns, kernel):
    JH, T = (8.0, 0.05) if L >= 16 else (4.0, 0.05)
    cfg = wl.Config(0, L, 1.0, JH, T, 0.0, "sphere", 0.0, 300 + L + B, M, K, B, ns)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
    ref = oracle.sweep_exact(L, 1.0, JH, T, 0.0, M, K, kernel, 4.0, S, ns, B, prop, uni, nthreads=16)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=T, n_energy=K, kernel=kernel, max_batch_sites=64, exact_batch_sites=max(B, 2))
    g.gfmc_set_spins(ctx, S)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_EXACT)
    out = g.gfmc_sweep(ctx, ns, B, prop, uni)
    S_gpu = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    margin = -ref["dS"] - np.log(uni)
    assert (np.abs(margin) > TIE).all(), "a decision fell inside the tie window; pick another seed"
    assert np.array_equal(out["accept"], ref["accept"])
    assert _ds_close(out["dS"], ref["dS"]).all(), np.abs(out["dS"] - ref["dS"]).max()
    assert np.array_equal(S_gpu, ref["spins"]) and np.array_equal(out["n_accepted"], ref["n_accepted"])
    assert np.abs(out["magnetization"] - ref["magnetization"]).max() < 1e-14
    if B == 1:      # one site per batch: nothing to correct, the exact mode is the sequential algorithm
        seq = oracle.sweep(L, 1.0, JH, T, 0.0, M, K, kernel, 4.0, S, ns, 1, prop, uni, nthreads=16)
        assert np.array_equal(out["accept"], seq["accept"]) and _ds_close(out["dS"], seq["dS"]).all()


def test_exact_run_and_device_pointers(oracle):
    """gfmc_run in exact mode == its replay through gfmc_sweep (host and device arrays)."""
    import torch
    L, M, B = 6, 16, 6
    S = wl.make_spins(L, seed=9)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=16, exact_batch_sites=8)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_EXACT)
    g.gfmc_set_spins(ctx, S)
    mag, nacc = g.gfmc_run(ctx, 17, 0, 2, B)
    S_run = g.gfmc_get_spins(ctx)
    P = np.stack([g.gfmc_random_proposals(ctx, 17, s)[0] for s in range(2)])
    U = np.stack([g.gfmc_random_proposals(ctx, 17, s)[1] for s in range(2)])
    g.gfmc_set_spins(ctx, S)
    r_h = g.gfmc_sweep(ctx, 2, B, P, U)
    assert np.array_equal(g.gfmc_get_spins(ctx), S_run) and np.array_equal(r_h["magnetization"], mag) and np.array_equal(r_h["n_accepted"], nacc)
    g.gfmc_set_spins(ctx, S)
    r_d = g.gfmc_sweep(ctx, 2, B, torch.from_numpy(P).cuda(), torch.from_numpy(U).cuda())
    for k in r_h:
        assert np.array_equal(r_d[k].cpu().numpy(), r_h[k]), k
    ref = oracle.sweep_exact(L, 1.0, 4.0, 0.1, 0.0, M, 2 * M, 0, 4.0, S, 2, B, P, U, nthreads=8)
    assert np.array_equal(r_h["accept"], ref["accept"]) and _ds_close(r_h["dS"], ref["dS"]).all()
    g.gfmc_destroy(ctx)


def test_exact_mode_validation():
    with pytest.raises(g.GfmcError, match="EINVAL"):
        g.gfmc_create(L=4, M=8, t=1.0, JH=4.0, T=0.1, max_batch_sites=8, exact_batch_sites=4, ph_symmetry=1)
    with pytest.raises(g.GfmcError, match="EINVAL"):
        g.gfmc_create(L=4, M=8, t=1.0, JH=0.0, T=0.1, max_batch_sites=8, exact_batch_sites=4, model=g.GFMC_MODEL_DEX_INF)
    with pytest.raises(g.GfmcError, match="EINVAL"):
        g.gfmc_create(L=4, M=8, t=1.0, JH=4.0, T=0.1, max_batch_sites=8, exact_batch_sites=9)
    ctx = g.gfmc_create(L=4, M=8, t=1.0, JH=4.0, T=0.1, max_batch_sites=8)
    with pytest.raises(g.GfmcError, match="ESTATE"):
        g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_EXACT)
    with pytest.raises(g.GfmcError, match="EINVAL"):
        g.gfmc_set_batch_mode(ctx, 7)
    g.gfmc_destroy(ctx)
    ctx = g.gfmc_create(L=4, M=8, t=1.0, JH=4.0, T=0.1, max_batch_sites=8, exact_batch_sites=4)
    S = wl.make_spins(4, seed=1)
    g.gfmc_set_spins(ctx, S)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_EXACT)
    with pytest.raises(g.GfmcError, match="exact_batch_sites"):
        g.gfmc_update_batch(ctx, np.arange(0, 10, 2, dtype=np.int32), S[:5], np.full(5, 0.5))
    with pytest.raises(g.GfmcError, match="exact_batch_sites"):
        g.gfmc_run(ctx, 1, 0, 1, 5)
    assert np.array_equal(g.gfmc_get_spins(ctx), S)
    g.gfmc_destroy(ctx)


def test_exact_batch_reports_non_finite_decisions_instead_of_rejecting_silently():
    """Device inputs are trusted, so a NaN can reach the exact-batch kernels (and a vanishing d_k would do the same through the
    Woodbury inverse).  -NaN > ln u is false: before this check such a batch quietly rejected every later site.  Now the call
    fails with GFMC_ESTATE and the configuration is untouched."""
    import torch
    L, M, n = 6, 16, 6
    S = wl.make_spins(L, seed=3)
    sites = wl.colour_sites(L, 0)[:n]
    prop = wl.make_spins(L, seed=4)[sites]
    prop[2, 0] = np.nan
    uni = np.full(n, 0.5)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=8, exact_batch_sites=8)
    g.gfmc_set_spins(ctx, S)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_EXACT)
    with pytest.raises(g.GfmcError, match="exact batch abandoned, configuration unchanged: non-finite Delta S") as ei:
        g.gfmc_update_batch(ctx, torch.from_numpy(sites).cuda(), torch.from_numpy(prop).cuda(), torch.from_numpy(uni).cuda())
    assert ei.value.code == -4
    assert np.array_equal(g.gfmc_get_spins(ctx), S)
    prop[2] = wl.make_spins(L, seed=4)[sites[2]]                       # the same batch without the NaN goes through on the same context
    dS, acc = g.gfmc_update_batch(ctx, sites, prop, uni)
    assert np.isfinite(dS).all()
    g.gfmc_destroy(ctx)
