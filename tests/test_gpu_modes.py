"""GPU parity tests (`-m gpu`) for the two further modes of the fused step, through the C ABI, against the oracle:
  * ph_symmetry = 1 (Eq. (1), one start vector per site) -- same moments / Delta S / decisions as the oracle;
  * model = GFMC_MODEL_DEX_INF (Eq. (2)-(3), (15)-(22)) against oracle/gfmc_oracle_dex.c.
Bars as in test_gpu_parity.py."""
import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl
from tests.dense import cheb_T

pytestmark = pytest.mark.gpu

MU_TOL = 1e-10
DS_RTOL = 1e-9
TIE = 1e-8


def _ds_close(a, b):
    return np.abs(a - b) <= DS_RTOL * np.maximum(1.0, np.abs(b))


# =========================================================================== particle-hole shortcut (Eq. (1))
@pytest.mark.parametrize("L,M,n,B", [
    (4, 64, 64, 64),      # every site of config 1's lattice, generic path, several slots per CTA
    (4, 16, 5, 2),        # chunking, odd site counts (last slot half empty)
    (2, 8, 8, 8),         # every neighbour reached twice (still bipartite)
    (6, 32, 51, 51),      # odd count, generic reduction
    (8, 256, 512, 512),   # config 2
    (16, 64, 301, 301),   # config 3 lattice, odd count
    (20, 24, 30, 30),
    (32, 32, 200, 200),   # config 4 lattice
    (64, 8, 5, 5),        # config 5 lattice
])
def test_ph_moments_match_oracle(oracle, L, M, n, B):
    JH = 8.0 if L >= 16 else 4.0
    S = wl.make_spins(L, seed=L)
    rng = np.random.default_rng(L * 1000 + M)
    sites = rng.choice(L ** 3, size=n, replace=False).astype(np.int32)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=0.05, max_batch_sites=B, ph_symmetry=1)
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments(ctx, sites)
    ref = oracle.moments_many(L, 1.0, JH, S, sites, M, nthreads=8)
    assert np.abs(mu - ref).max() <= MU_TOL
    nvec, _ = g.gfmc_last_step_loop_vectors(ctx)
    assert nvec == min(B, n if n <= B else n % B or B)            # ONE start vector per site of the last chunk
    g.gfmc_destroy(ctx)


def test_ph_rejects_odd_L():
    with pytest.raises(g.GfmcError):
        g.gfmc_create(L=5, M=8, t=1.0, JH=4.0, T=0.1, max_batch_sites=4, ph_symmetry=1)


def test_ph_sweep_matches_oracle_and_two_vector_path(oracle):
    cfg = wl.CONFIGS[2]
    L, M, K, B, ns = cfg.L, 32, 64, 100, 2
    S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
    ref = oracle.sweep(L, cfg.t, cfg.JH, cfg.T, 0.0, M, K, 0, 4.0, S, ns, B, prop, uni, nthreads=8)
    outs = []
    for ph in (1, 0):
        ctx = g.gfmc_create(L=L, M=M, t=cfg.t, JH=cfg.JH, T=cfg.T, n_energy=K, max_batch_sites=B, ph_symmetry=ph)
        g.gfmc_set_spins(ctx, S)
        out = g.gfmc_sweep(ctx, ns, B, prop, uni)
        out["spins"] = g.gfmc_get_spins(ctx)
        outs.append(out)
        g.gfmc_destroy(ctx)
    out = outs[0]
    # sweep 0 is evaluated on identical configurations: strict parity; later sweeps only while no decision was a tie
    assert _ds_close(out["dS"][0], ref["dS"][0]).all()
    margin = -ref["dS"] - np.log(uni)
    assert (np.abs(margin) > TIE).all()
    assert np.array_equal(out["accept"], ref["accept"])
    assert _ds_close(out["dS"], ref["dS"]).all()
    assert np.array_equal(out["spins"], ref["spins"])
    assert np.array_equal(out["n_accepted"], ref["n_accepted"])
    assert np.abs(out["magnetization"] - ref["magnetization"]).max() < 1e-14
    assert np.array_equal(out["accept"], outs[1]["accept"]) and _ds_close(out["dS"], outs[1]["dS"]).all()


# =========================================================================== J_H -> infinity (Eq. (2)-(3), (15)-(22))
def _dex_ctx(L, M, B, T=0.05, K=0, t=1.0, kernel=0, **kw):
    return g.gfmc_create(L=L, M=M, t=t, JH=0.0, T=T, n_energy=K, kernel=kernel, max_batch_sites=B, model=g.GFMC_MODEL_DEX_INF, **kw)


@pytest.mark.parametrize("L,kind,cone", [(4, "sphere", 0.0), (7, "sphere", 0.0), (8, "cone", 0.3)])
def test_dex_hopping_matches_oracle(oracle, L, kind, cone):
    S = wl.make_spins(L, seed=40 + L, kind=kind, cone=cone)
    S[3] = [0.0, 0.0, 1.0]; S[4] = [0.0, 0.0, -1.0]; S[5] = [-1.0, 0.0, 0.0]       # poles and the atan2 branch cut
    ctx = _dex_ctx(L, 8, 1)
    g.gfmc_set_spins(ctx, S)
    Tb = g.gfmc_hopping(ctx)
    a, b = g.gfmc_bounds(ctx)
    assert (a, b) == oracle.dex_bounds(1.0)
    N = L ** 3
    idx = np.arange(N); x, y, z = idx % L, (idx // L) % L, idx // (L * L)
    nbr = [((x + 1) % L) + L * (y + L * z), x + L * (((y + 1) % L) + L * z), x + L * (y + L * ((z + 1) % L))]
    for d in range(3):
        ref = np.array([oracle.dex_hopping(S[i], S[nbr[d][i]]) for i in range(N)])
        assert np.abs(Tb[d] - ref).max() < 1e-14
    g.gfmc_destroy(ctx)


@pytest.mark.parametrize("L,M,n,B,t", [
    (4, 64, 64, 64, 1.0),     # all sites, generic path
    (3, 16, 27, 27, 0.7),     # odd L, generic reduction, neighbours of o adjacent to each other
    (5, 16, 7, 3, 1.0),       # chunking with odd counts
    (6, 32, 51, 51, 1.0),     # the paper's smallest lattice
    (8, 256, 256, 256, 1.0),
    (16, 64, 301, 301, 1.3),
    (20, 24, 30, 30, 1.0),    # the paper's 20^3
    (32, 32, 200, 200, 1.0),  # the paper's largest lattice
    (64, 8, 5, 5, 1.0),
])
def test_dex_moments_match_oracle(oracle, L, M, n, B, t):
    S = wl.make_spins(L, seed=L + 1)
    rng = np.random.default_rng(L * 1000 + M)
    sites = rng.choice(L ** 3, size=n, replace=False).astype(np.int32)
    prop = wl.make_spins(L, seed=L + 2)[sites]
    ctx = _dex_ctx(L, M, B, t=t)
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments_ov(ctx, sites, prop)
    ref = oracle.dex_moments_many(L, t, S, sites, prop, M, nthreads=8)
    scale = np.maximum(1.0, np.abs(ref[:, 0, 1, 1].real))[:, None, None, None]     # |v| is not normalised: <v|v> <= 24 t^2
    assert (np.abs(mu - ref) / scale).max() <= MU_TOL
    assert np.array_equal(mu[:, :, 1, 0], mu[:, :, 0, 1].conj())
    with pytest.raises(g.GfmcError):
        g.gfmc_moments(ctx, sites)
    g.gfmc_destroy(ctx)


@pytest.mark.parametrize("mode", ["dex", "ph"])
@pytest.mark.parametrize("L,M,n", [(4, 32, 33), (6, 24, 51), (8, 32, 200), (10, 16, 41), (12, 12, 30)])
def test_streaming_kernel_on_small_lattices_other_modes(oracle, mode, L, M, n):
    """L <= 12 runs the shared-memory-resident kernel in every mode; flags = GFMC_FLAG_NO_RESIDENT sends the same lattices through the
    streaming kernel.  Both must match the oracle and each other (J_H->inf and one-vector modes; Eq. (1) default: test_gpu_parity)."""
    S = wl.make_spins(L, seed=L + 21)
    sites = np.random.default_rng(L + 5).choice(L ** 3, size=n, replace=False).astype(np.int32)
    prop = wl.make_spins(L, seed=L + 22)[sites]
    if mode == "dex":
        ref = oracle.dex_moments_many(L, 1.0, S, sites, prop, M, nthreads=8)
        scale = np.maximum(1.0, np.abs(ref[:, 0, 1, 1].real))[:, None, None, None]
    else:
        ref = oracle.moments_many(L, 1.0, 4.0, S, sites, M, nthreads=8)
        scale = 1.0
    got = {}
    for flag in ("1", "0"):
        fl = g.GFMC_FLAG_NO_RESIDENT if flag == "1" else 0
        ctx = _dex_ctx(L, M, n, flags=fl) if mode == "dex" else g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.05, max_batch_sites=n, ph_symmetry=1, flags=fl)
        g.gfmc_set_spins(ctx, S)
        got[flag] = g.gfmc_moments_ov(ctx, sites, prop) if mode == "dex" else g.gfmc_moments(ctx, sites)
        assert g.gfmc_launch_counts(ctx)[0] == (M // 2 if flag == "1" else 1)
        g.gfmc_destroy(ctx)
        assert (np.abs(got[flag] - ref) / scale).max() <= MU_TOL
    assert (np.abs(got["0"] - got["1"]) / scale).max() <= 1e-13


@pytest.mark.parametrize("L", [32, 64])
def test_dex_ferromagnet_band_large_lattices(L):
    """Aligned spins: t_ij = 1, mu_n(o,o) = L^-3 sum_k T_n(eps_k / 6t) (free band) at full-size lattices, no oracle."""
    M, P = 64, 6
    S = wl.ferromagnet(L, (0.3, -0.5, 0.81))
    sites = np.random.default_rng(2).choice(L ** 3, size=P, replace=False).astype(np.int32)
    ctx = _dex_ctx(L, M, P)
    g.gfmc_set_spins(ctx, S)
    mu = g.gfmc_moments_ov(ctx, sites, wl.make_spins(2, seed=3)[:P])
    k = 2 * np.pi * np.arange(L) / L
    eps = (-2.0 * (np.cos(k)[:, None, None] + np.cos(k)[None, :, None] + np.cos(k)[None, None, :])).ravel()
    ref = np.array([cheb_T(n, eps / 6.0).mean() for n in range(M)])
    assert np.abs(mu[:, :, 0, 0] - ref[None]).max() <= MU_TOL
    g.gfmc_destroy(ctx)


@pytest.mark.parametrize("kernel", [0, 1])
def test_dex_green_and_delta_S_match_oracle(oracle, kernel):
    L, M, K, T = 6, 64, 128, 0.05
    S = wl.make_spins(L, seed=12)
    sites = np.array([0, 21, 100, 215, 7], dtype=np.int32)
    prop = wl.make_spins(L, seed=13)[sites]
    ctx = _dex_ctx(L, M, 4, T=T, K=K, kernel=kernel)
    g.gfmc_set_spins(ctx, S)
    E, G = g.gfmc_local_green_ov(ctx, sites, prop)
    dS = g.gfmc_delta_S(ctx, sites, prop)
    a, b = g.gfmc_bounds(ctx)
    for j, s in enumerate(sites):
        mu = oracle.dex_moments(L, 1.0, S, int(s), prop[j], M)
        Eo, Gt = oracle.green(mu, K, kernel, 4.0, a, b)
        assert np.abs(E - Eo).max() < 1e-13
        assert np.abs(G[j] - Gt / a).max() <= 1e-10 * np.abs(Gt / a).max()
        ref = oracle.dex_site_dS(L, 1.0, T, 0.0, M, K, kernel, 4.0, S, int(s), prop[j])
        assert _ds_close(dS[j], ref), (j, dS[j], ref)
    assert np.array_equal(g.gfmc_get_spins(ctx), S)
    g.gfmc_destroy(ctx)


@pytest.mark.parametrize("L,M,B,ns", [(4, 32, 1, 1), (4, 32, 9, 2), (8, 32, 100, 2)])
def test_dex_sweep_matches_oracle(oracle, L, M, B, ns):
    cfg = wl.CONFIGS[1] if L == 4 else wl.CONFIGS[2]
    K, T = 2 * M, 0.05
    S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
    ref = oracle.dex_sweep(L, 1.0, T, 0.0, M, K, 0, 4.0, S, ns, B, prop, uni, nthreads=8)
    ctx = _dex_ctx(L, M, B, T=T, K=K)
    g.gfmc_set_spins(ctx, S)
    out = g.gfmc_sweep(ctx, ns, B, prop, uni)
    margin = -ref["dS"] - np.log(uni)
    assert (np.abs(margin) > TIE).all()
    assert np.array_equal(out["accept"], ref["accept"])
    assert _ds_close(out["dS"], ref["dS"]).all()
    assert np.array_equal(g.gfmc_get_spins(ctx), ref["spins"])
    assert np.array_equal(out["n_accepted"], ref["n_accepted"])
    assert np.abs(out["magnetization"] - ref["magnetization"]).max() < 1e-14
    assert 0 < out["n_accepted"].sum() < ns * L ** 3
    g.gfmc_destroy(ctx)


def test_dex_update_batch_device_pointers(oracle):
    import torch
    L, M, K, T = 8, 32, 64, 0.05
    cfg = wl.CONFIGS[2]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(L, 1)[:77]
    ctx = _dex_ctx(L, M, 128, T=T, K=K)
    g.gfmc_set_spins(ctx, torch.from_numpy(S).cuda())
    dS, acc = g.gfmc_update_batch(ctx, torch.from_numpy(sites).cuda(), torch.from_numpy(prop[0][sites]).cuda(),
                                  torch.from_numpy(uni[0][sites]).cuda())
    dS, acc = dS.cpu().numpy(), acc.cpu().numpy()
    ref = np.array([oracle.dex_site_dS(L, 1.0, T, 0.0, M, K, 0, 4.0, S, int(s), prop[0][s]) for s in sites])
    assert _ds_close(dS, ref).all()
    margin = -ref - np.log(uni[0][sites])
    clear = np.abs(margin) > TIE
    assert np.array_equal(acc[clear], (margin > 0).astype(np.uint8)[clear])
    S2 = S.copy(); S2[sites[acc.astype(bool)]] = prop[0][sites[acc.astype(bool)]]
    assert np.array_equal(g.gfmc_get_spins(ctx), S2)
    # the bond amplitudes follow the accepted flips ("update H", Alg. 1 line 12)
    Tb = g.gfmc_hopping(ctx)
    i = int(sites[np.flatnonzero(acc)[0]])
    assert abs(Tb[0][i] - oracle.dex_hopping(S2[i], S2[(i % L + 1) % L + L * (i // L)])) < 1e-14
    g.gfmc_destroy(ctx)


# =========================================================================== two Chebyshev steps per pass (temporal blocking, f2)
@pytest.mark.parametrize("M,n", [(32, 200), (16, 301), (8, 3), (64, 148)])
def test_two_step_moments_match_oracle_and_single_step(oracle, M, n):
    """flags = GFMC_FLAG_TWO_STEP (one-vector mode, L = 32): r_m and r_{m+1} in one pass over the vectors, the intermediate planes in shared
    memory.  Same moments as the oracle's plain two-vector recursion and as the one-step-per-launch kernel; half the launches."""
    L, JH = 32, 8.0
    S = wl.make_spins(L, seed=77)
    sites = np.random.default_rng(M + n).choice(L ** 3, size=n, replace=False).astype(np.int32)
    got = {}
    for two in (1, 0):
        ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=0.05, max_batch_sites=n, ph_symmetry=1, flags=g.GFMC_FLAG_TWO_STEP if two else 0)
        g.gfmc_set_spins(ctx, S)
        a = g.gfmc_moments(ctx, sites)
        b = g.gfmc_moments(ctx, sites)
        assert np.array_equal(a, b)                                    # fixed summation order: bit-reproducible
        assert g.gfmc_launch_counts(ctx)[0] == 2 * (M // 4 if two else M // 2)
        got[two] = a
        g.gfmc_destroy(ctx)
    sub = np.arange(0, n, max(1, n // 10))
    ref = oracle.moments_many(L, 1.0, JH, S, sites[sub], M, nthreads=8)
    assert np.abs(got[1][sub] - ref).max() <= MU_TOL
    assert np.abs(got[1] - got[0]).max() <= 1e-13


def test_two_step_update_batch_and_validation(oracle):
    L, M, K, n = 32, 32, 64, 64
    cfg = wl.CONFIGS[4]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(L, 1)[100:100 + n]
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=8.0, T=0.02, n_energy=K, max_batch_sites=n, ph_symmetry=1, flags=g.GFMC_FLAG_TWO_STEP)
    g.gfmc_set_spins(ctx, S)
    dS, acc = g.gfmc_update_batch(ctx, sites, prop[0][sites], uni[0][sites])
    ref = np.array([oracle.site_dS(L, 1.0, 8.0, 0.02, 0.0, M, K, 0, 4.0, S, int(s), prop[0][s]) for s in sites[::8]])
    assert _ds_close(dS[::8], ref).all()
    margin = -ref - np.log(uni[0][sites[::8]])
    clear = np.abs(margin) > TIE
    assert np.array_equal(acc[::8][clear], (margin > 0).astype(np.uint8)[clear])
    nvec, nbytes = g.gfmc_last_step_loop_vectors(ctx)
    assert nvec == n and g.gfmc_last_step_loop_ms(ctx)[1] == M // 2       # fused STEPS, two per launch
    g.gfmc_destroy(ctx)
    for bad in (dict(L=16, M=32, ph_symmetry=1), dict(L=32, M=30, ph_symmetry=1), dict(L=32, M=32, ph_symmetry=0)):
        with pytest.raises(g.GfmcError, match="EINVAL"):
            g.gfmc_create(t=1.0, JH=8.0, T=0.05, max_batch_sites=4, flags=g.GFMC_FLAG_TWO_STEP, **bad)
