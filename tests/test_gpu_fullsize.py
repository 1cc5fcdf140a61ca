"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (`-m gpu`).

The oracle cannot finish a whole batch at these sizes, so (SURVEY.md §8(c) "at scale"): the CUDA path runs the
full batch; the oracle re-evaluates a SAMPLE of its sites one by one against the same (frozen) configuration;
full-batch outputs are additionally checked through properties that hold at any size (closed-form ferromagnet
moments, Hermiticity, mu_0, |mu| <= 1)."""
import os

import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl
from tests.dense import SIGMA, cheb_T

pytestmark = pytest.mark.gpu

NTH = max(1, min(16, os.cpu_count() or 1))


def _sample_check(oracle, cfg, S, sites, prop_s, uni_s, dS, acc, sample, M, K):
    ref = np.array([0.0] * len(sample))
    mus = oracle.moments_many(cfg.L, cfg.t, cfg.JH, S, sites[sample], M, nthreads=NTH)
    a, b = oracle.bounds(cfg.t, cfg.JH)
    for j, idx in enumerate(sample):
        s = int(sites[idx])
        _, Gt = oracle.green(mus[j], K, 0, 4.0, a, b)
        ref[j] = oracle.delta_S(Gt, S[s], prop_s[s], cfg.JH, a, b, cfg.T, cfg.mu)
    got = dS[sample]
    assert np.all(np.abs(got - ref) <= 1e-9 * np.maximum(1.0, np.abs(ref))), (got, ref)
    margin = -ref - np.log(uni_s[sites[sample]])
    clear = np.abs(margin) > 1e-8
    assert np.array_equal(acc[sample][clear], (margin > 0).astype(np.uint8)[clear])
    return mus


def test_config4_full_batch_L32_M1024_B2048(oracle):
    """The headline configuration: L=32, J_H=8, T=0.02, M=1024, K=2048, 2048-site checkerboard batch (4096 start
    vectors).  One frozen-batch update through gfmc_update_batch; oracle on 6 sampled sites."""
    cfg = wl.CONFIGS[4]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[:cfg.batch_sites]
    ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=cfg.JH, T=cfg.T, n_energy=cfg.K, max_batch_sites=cfg.batch_sites)
    g.gfmc_set_spins(ctx, S)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop[0][sites], uni[0][sites])
    ms, steps = g.gfmc_last_step_loop_ms(ctx)
    assert steps == cfg.M // 2
    S_after = g.gfmc_get_spins(ctx)
    S_ref = S.copy(); S_ref[sites[acc == 1]] = prop[0][sites[acc == 1]]
    assert np.array_equal(S_after, S_ref)
    assert np.isfinite(dS).all() and 0 < acc.sum() < len(sites)
    sample = np.array([0, 1, 777, 1024, 2046, 2047])
    _sample_check(oracle, cfg, S, sites, prop[0], uni[0], dS, acc, sample, cfg.M, cfg.K)
    g.gfmc_destroy(ctx)


def test_config3_full_batch_L16_M512_B512(oracle):
    cfg = wl.CONFIGS[3]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 1)[-cfg.batch_sites:]
    ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=cfg.JH, T=cfg.T, n_energy=cfg.K, max_batch_sites=cfg.batch_sites)
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments(ctx, sites)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop[0][sites], uni[0][sites])
    sample = np.arange(0, cfg.batch_sites, 37)
    mus = _sample_check(oracle, cfg, S, sites, prop[0], uni[0], dS, acc, sample, cfg.M, cfg.K)
    assert np.abs(mu[sample] - mus).max() <= 1e-10
    assert np.abs(mu).max() <= 1 + 1e-12 and np.array_equal(mu[:, :, 1, 0], mu[:, :, 0, 1].conj())
    g.gfmc_destroy(ctx)


def test_config4_lattice_moment_prefix_full_batch(oracle):
    """Moments do not depend on M: the first 128 moments of a full 2048-site launch equal the oracle's M=128 run."""
    cfg = wl.CONFIGS[4]
    S, _, _ = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 1)[:cfg.batch_sites]
    ctx = g.gfmc_create(L=cfg.L, M=128, t=cfg.t, JH=cfg.JH, T=cfg.T, max_batch_sites=cfg.batch_sites)
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments(ctx, sites)
    sample = np.array([0, 5, 1000, 2047])
    ref = oracle.moments_many(cfg.L, cfg.t, cfg.JH, S, sites[sample], 128, nthreads=NTH)
    assert np.abs(mu[sample] - ref).max() <= 1e-10
    assert np.abs(mu).max() <= 1 + 1e-12
    g.gfmc_destroy(ctx)


def test_config5_lattice_L64_large_batch(oracle):
    """L=64 (D = 524288): a 1024-site batch (2048 start vectors, 32 GiB of work vectors, well beyond L2) in the cone
    configuration of config 5; oracle on 2 sampled sites for the first 64 moments, closed-form ferromagnet for all."""
    cfg = wl.CONFIGS[5]
    B, M = 1024, 64
    S, _, _ = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[::128][:B].copy()
    try:
        ctx = g.gfmc_create(L=cfg.L, M=M, t=cfg.t, JH=cfg.JH, T=cfg.T, max_batch_sites=B)
    except g.GfmcError as e:          # a smaller device: say so instead of passing silently
        pytest.skip(f"not enough device memory for the L=64 batch: {e}")
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments(ctx, sites)
    sample = np.array([0, B - 1])
    ref = oracle.moments_many(cfg.L, cfg.t, cfg.JH, S, sites[sample], M, nthreads=2)
    assert np.abs(mu[sample] - ref).max() <= 1e-10
    # ferromagnet along a tilted axis: closed form for every site of the batch
    nhat = np.array([0.6, 0.0, 0.8])
    g.gfmc_set_spins(ctx, wl.ferromagnet(cfg.L, nhat))
    mu = g.gfmc_moments(ctx, sites)
    a, _ = g.gfmc_bounds(ctx)
    k = 2 * np.pi * np.arange(cfg.L) / cfg.L
    eps = (-2 * cfg.t * (np.cos(k)[:, None, None] + np.cos(k)[None, :, None] + np.cos(k)[None, None, :])).ravel()
    mp = np.array([cheb_T(n, (eps + cfg.JH) / a).mean() for n in range(M)])
    mm = np.array([cheb_T(n, (eps - cfg.JH) / a).mean() for n in range(M)])
    nsig = np.einsum("c,cab->ab", nhat, SIGMA)
    refF = mp[:, None, None] * (np.eye(2) + nsig) / 2 + mm[:, None, None] * (np.eye(2) - nsig) / 2
    assert np.abs(mu - refF[None]).max() <= 1e-10
    g.gfmc_destroy(ctx)


def test_config4_ph_symmetry_full_batch(oracle):
    """Config 4 with ph_symmetry = 1 (one start vector per site; the launch configuration bench.py's `modes.ph_symmetry`
    times): full 2048-site batch, oracle (plain two-vector recursion) on sampled sites."""
    cfg = wl.CONFIGS[4]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[:cfg.batch_sites]
    ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=cfg.JH, T=cfg.T, n_energy=cfg.K, max_batch_sites=cfg.batch_sites,
                        ph_symmetry=1)
    g.gfmc_set_spins(ctx, S)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop[0][sites], uni[0][sites])
    nvec, nbytes = g.gfmc_last_step_loop_vectors(ctx)
    assert nvec == cfg.batch_sites and nbytes == 48 * cfg.batch_sites * cfg.D
    S_ref = S.copy(); S_ref[sites[acc == 1]] = prop[0][sites[acc == 1]]
    assert np.array_equal(g.gfmc_get_spins(ctx), S_ref)
    sample = np.array([0, 1, 1023, 1024, 2047])
    _sample_check(oracle, cfg, S, sites, prop[0], uni[0], dS, acc, sample, cfg.M, cfg.K)
    g.gfmc_destroy(ctx)


def test_L32_dex_full_batch_M1024_B2048(oracle):
    """The paper's own Hamiltonian (Eq. (2)-(3)) at its largest lattice 32^3, M = 1024, K = 2048, 2048-site
    batch (4096 start vectors |o>, |v>): the launch configuration of bench.py's `modes.dex_inf`; oracle on sampled sites."""
    cfg = wl.CONFIGS[4]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[:cfg.batch_sites]
    ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=0.0, T=cfg.T, n_energy=cfg.K, max_batch_sites=cfg.batch_sites,
                        model=g.GFMC_MODEL_DEX_INF)
    g.gfmc_set_spins(ctx, S)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop[0][sites], uni[0][sites])
    nvec, nbytes = g.gfmc_last_step_loop_vectors(ctx)
    assert nvec == 2 * cfg.batch_sites and nbytes == 48 * 2 * cfg.batch_sites * cfg.N
    S_ref = S.copy(); S_ref[sites[acc == 1]] = prop[0][sites[acc == 1]]
    assert np.array_equal(g.gfmc_get_spins(ctx), S_ref)
    assert np.isfinite(dS).all() and 0 < acc.sum() < len(sites)
    sample = np.array([0, 1023, 2047])       # (the J_H->inf oracle costs ~45 s per site at M = 1024)
    ref = np.array([oracle.dex_site_dS(cfg.L, cfg.t, cfg.T, cfg.mu, cfg.M, cfg.K, 0, 4.0, S, int(sites[j]), prop[0][sites[j]])
                    for j in sample])
    assert np.all(np.abs(dS[sample] - ref) <= 1e-9 * np.maximum(1.0, np.abs(ref))), (dS[sample], ref)
    margin = -ref - np.log(uni[0][sites[sample]])
    clear = np.abs(margin) > 1e-8
    assert np.array_equal(acc[sample][clear], (margin > 0).astype(np.uint8)[clear])
    g.gfmc_destroy(ctx)


def _ferromagnet_moments(L, t, JH, a, M, nhat):
    """Closed form for aligned spins along nhat (SURVEY.md §8(c) pin iii): mu_n = mu+_n P+ + mu-_n P-,
    mu^+-_n = L^-3 sum_k T_n((eps_k +- J_H)/a), eps_k = -2t (cos kx + cos ky + cos kz), P+- = (1 +- nhat.sigma)/2."""
    k = 2 * np.pi * np.arange(L) / L
    eps = (-2 * t * (np.cos(k)[:, None, None] + np.cos(k)[None, :, None] + np.cos(k)[None, None, :])).ravel()
    mp = np.array([cheb_T(n, (eps + JH) / a).mean() for n in range(M)])
    mm = np.array([cheb_T(n, (eps - JH) / a).mean() for n in range(M)])
    nsig = np.einsum("c,cab->ab", np.asarray(nhat), SIGMA)
    return mp[:, None, None] * (np.eye(2) + nsig) / 2 + mm[:, None, None] * (np.eye(2) - nsig) / 2


def test_config5_full_batch_L64_M2048_B4096(oracle):
    """Config 5 exactly as BASELINE.json states it: L=64 (D = 524288), J_H=8, T=0.01, cone spins, M=2048, K=4096, a 4096-site
    checkerboard batch (8192 start vectors, 128 GiB of work vectors, 1024 fused-step launches, the direct-sum Green kernel).
    gfmc_moments and gfmc_update_batch on the full batch; the oracle re-evaluates 4 sampled sites: all 2048 moments,
    Delta S and the decisions."""
    cfg = wl.CONFIGS[5]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[:cfg.batch_sites]
    try:
        ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=cfg.JH, T=cfg.T, n_energy=cfg.K, max_batch_sites=cfg.batch_sites)
    except (g.GfmcError, RuntimeError) as e:      # GFMC_ENOMEM / torch OOM on a smaller device: say so instead of passing silently
        pytest.skip(f"not enough device memory for config 5 (128 GiB of work vectors): {e}")
    g.gfmc_set_spins(ctx, S)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop[0][sites], uni[0][sites])
    ms, steps = g.gfmc_last_step_loop_ms(ctx)
    assert steps == cfg.M // 2
    S_after = g.gfmc_get_spins(ctx)
    S_ref = S.copy(); S_ref[sites[acc == 1]] = prop[0][sites[acc == 1]]
    assert np.array_equal(S_after, S_ref)
    assert np.isfinite(dS).all() and 0 < acc.sum() < len(sites)
    sample = np.array([0, 1365, 2730, 4095])
    mus = _sample_check(oracle, cfg, S, sites, prop[0], uni[0], dS, acc, sample, cfg.M, cfg.K)
    # moments of the same sites from the same launch shape (full batch, configuration restored first)
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments(ctx, sites)
    err = np.abs(mu[sample] - mus).max()
    assert err <= 1e-10, err
    assert np.abs(mu).max() <= 1 + 1e-12 and np.array_equal(mu[:, :, 1, 0], mu[:, :, 0, 1].conj())
    g.gfmc_destroy(ctx)


def test_config4_ferromagnet_closed_form_full_batch():
    """Every site of the headline launch shape (L=32, 2048-site batch = 4096 start vectors) against the textbook band of the
    ferromagnet along a tilted axis: pins all 2048 slots of a full batch without oracle time."""
    cfg = wl.CONFIGS[4]
    M = 64
    nhat = np.array([0.48, -0.6, 0.64])
    sites = wl.colour_sites(cfg.L, 1)[-cfg.batch_sites:]
    ctx = g.gfmc_create(L=cfg.L, M=M, t=cfg.t, JH=cfg.JH, T=cfg.T, max_batch_sites=cfg.batch_sites)
    g.gfmc_set_spins(ctx, wl.ferromagnet(cfg.L, nhat))
    mu = g.gfmc_moments(ctx, sites)
    a, _ = g.gfmc_bounds(ctx)
    g.gfmc_destroy(ctx)
    ref = _ferromagnet_moments(cfg.L, cfg.t, cfg.JH, a, M, nhat)
    assert np.abs(mu - ref[None]).max() <= 1e-10


@pytest.mark.parametrize("L,M,P", [(96, 12, 6), (128, 10, 4), (256, 6, 2)])
def test_largest_lattices_the_header_allows(oracle, L, M, P):
    """include/gfmc.h promises 2 <= L <= 256.  L = 96, 128, 256 run the run-time-L kernel with Ty = 5, 4, 2 rows + 2 halo rows
    per stage and the CTA-wide R_prev ring: tiny batch, ferromagnet closed form for every site + the oracle on 2 sites of a
    random configuration."""
    t, JH = 1.0, 8.0
    nhat = np.array([0.6, 0.0, 0.8])
    rng = np.random.default_rng(L)
    sites = rng.choice(L ** 3, size=P, replace=False).astype(np.int32)
    sites[0] = 0; sites[-1] = L ** 3 - 1                  # the periodic wrap in all three directions
    try:
        ctx = g.gfmc_create(L=L, M=M, t=t, JH=JH, T=0.05, max_batch_sites=P)
    except (g.GfmcError, RuntimeError) as e:
        pytest.skip(f"not enough device memory for L={L}: {e}")
    g.gfmc_set_spins(ctx, wl.ferromagnet(L, nhat))
    mu = g.gfmc_moments(ctx, sites)
    a, _ = g.gfmc_bounds(ctx)
    assert np.abs(mu - _ferromagnet_moments(L, t, JH, a, M, nhat)[None]).max() <= 1e-10
    S = wl.make_spins(L, seed=L)
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments(ctx, sites)
    ref = oracle.moments_many(L, t, JH, S, sites[[0, -1]], M, nthreads=2)
    assert np.abs(mu[[0, -1]] - ref).max() <= 1e-10
    g.gfmc_destroy(ctx)


def test_config4_two_step_full_batch(oracle):
    """Config 4 with ph_symmetry = 1 and two Chebyshev steps per pass (the launch configuration of bench.py's `modes.ph_two_step`): full
    2048-site batch, M = 1024 (256 passes), oracle (plain two-vector recursion, one step at a time) on sampled sites."""
    cfg = wl.CONFIGS[4]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[:cfg.batch_sites]
    ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=cfg.JH, T=cfg.T, n_energy=cfg.K, max_batch_sites=cfg.batch_sites,
                        ph_symmetry=1, flags=g.GFMC_FLAG_TWO_STEP)
    g.gfmc_set_spins(ctx, S)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop[0][sites], uni[0][sites])
    assert g.gfmc_launch_counts(ctx)[0] == cfg.M // 4
    S_ref = S.copy(); S_ref[sites[acc == 1]] = prop[0][sites[acc == 1]]
    assert np.array_equal(g.gfmc_get_spins(ctx), S_ref)
    sample = np.array([0, 1, 1023, 1024, 2047])
    _sample_check(oracle, cfg, S, sites, prop[0], uni[0], dS, acc, sample, cfg.M, cfg.K)
    g.gfmc_destroy(ctx)
