"""the Algorithm-1 driver with device-side trial moves (gfmc_random_proposals / gfmc_run) against the oracle's
own Philox generator (oracle/rng.py) feeding the oracle's sweep."""
import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def oracle():
    from oracle import oracle as o
    o.build()
    return o


@pytest.mark.parametrize("L,seed,sweep", [(4, 1, 0), (8, 2**40 + 17, 5), (16, 123456789, 2**33 + 1)])
def test_random_proposals_match_the_oracle_generator(L, seed, sweep):
    from oracle import rng
    ctx = g.gfmc_create(L=L, M=8, t=1.0, JH=4.0, T=0.05, max_batch_sites=1)
    prop, uni = g.gfmc_random_proposals(ctx, seed, sweep)
    pd, ud = g.gfmc_random_proposals(ctx, seed, sweep, device=True)
    g.gfmc_destroy(ctx)
    pr, ur = rng.proposals(seed, sweep, L ** 3)
    assert np.array_equal(uni, ur)                       # integer work + one exact subtraction: bit-exact
    assert np.array_equal(prop[:, 2], pr[:, 2])          # z = 2 u1 - 1 is exact
    assert np.abs(prop - pr).max() <= 4e-16              # sin/cos of two libraries: a few ulp
    assert np.array_equal(pd.cpu().numpy(), prop) and np.array_equal(ud.cpu().numpy(), uni)


@pytest.mark.parametrize("L,M,K,B,ph", [(4, 32, 64, 1, 0), (4, 32, 64, 8, 0), (6, 24, 48, 20, 1), (8, 16, 32, 64, 0)])
def test_run_matches_oracle_chain(oracle, L, M, K, B, ph):
    """gfmc_run == oracle sweeps fed by the oracle's generator: decisions identical away from ties, spins equal to a few ulp
    (the trial spins themselves differ by sin/cos rounding), magnetization and acceptance counts equal."""
    from oracle import rng
    JH, T, seed, first, n = 4.0, 0.05, 77 + L, 3, 2
    S = wl.make_spins(L, seed=90 + L)
    fn = lambda S_, p, u: oracle.sweep(L, 1.0, JH, T, 0.0, M, K, 0, 4.0, S_, 1, B, p, u, nthreads=8)
    ref = rng.run_chain(fn, S, seed, first, n)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=T, n_energy=K, max_batch_sites=B, ph_symmetry=ph)
    g.gfmc_set_spins(ctx, S)
    mag, nacc = g.gfmc_run(ctx, seed, first, n, B)
    S_gpu = g.gfmc_get_spins(ctx)
    # replay the same chain through gfmc_sweep with the library's own numbers: must be the same chain bit for bit
    g.gfmc_set_spins(ctx, S)
    P = np.stack([g.gfmc_random_proposals(ctx, seed, first + s)[0] for s in range(n)])
    U = np.stack([g.gfmc_random_proposals(ctx, seed, first + s)[1] for s in range(n)])
    r2 = g.gfmc_sweep(ctx, n, B, P, U)
    dS2, acc2, mag2, nacc2 = r2["dS"], r2["accept"], r2["magnetization"], r2["n_accepted"]
    S_replay = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    assert np.array_equal(S_replay, S_gpu) and np.array_equal(mag2, mag) and np.array_equal(nacc2, nacc)
    margin = -ref["dS"] - np.log(ref["uniforms"])
    clear = np.abs(margin) > 1e-8
    assert clear.mean() > 0.99
    assert np.array_equal(acc2[clear], ref["accept"][clear])
    assert np.abs(dS2 - ref["dS"]).max() <= 1e-9 * max(1.0, np.abs(ref["dS"]).max())
    if clear.all():
        assert np.array_equal(nacc, ref["n_accepted"])
        assert np.abs(S_gpu - ref["spins"]).max() <= 4e-16
        assert np.abs(mag - ref["magnetization"]).max() <= 1e-14


def test_run_is_resumable_and_validates():
    """(spins, seed, next sweep) is a complete checkpoint: 3 sweeps == 1 sweep + 2 sweeps; bad arguments are refused."""
    L, M, B = 4, 16, 8
    S = wl.make_spins(L, seed=5)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=B)
    with pytest.raises(g.GfmcError):
        g.gfmc_run(ctx, 1, 0, 1, B)                       # spins not set
    g.gfmc_set_spins(ctx, S)
    m3, n3 = g.gfmc_run(ctx, 9, 0, 3, B)
    Sa = g.gfmc_get_spins(ctx)
    g.gfmc_set_spins(ctx, S)
    m1, n1 = g.gfmc_run(ctx, 9, 0, 1, B)
    m2, n2 = g.gfmc_run(ctx, 9, 1, 2, B)
    assert np.array_equal(g.gfmc_get_spins(ctx), Sa)
    assert np.array_equal(np.concatenate([m1, m2]), m3) and np.array_equal(np.concatenate([n1, n2]), n3)
    with pytest.raises(g.GfmcError):
        g.gfmc_run(ctx, 1, 0, 1, B + 1)
    with pytest.raises(g.GfmcError):
        g.gfmc_run(ctx, 1, -1, 1, B)
    g.gfmc_destroy(ctx)


def test_magnetization_curve_driver_matches_oracle_chain(oracle):
    """The host driver (annealing through two temperatures on one chain) == the oracle run with the same sweep indices."""
    from oracle import rng
    from paper_1303_6016_b200 import driver
    L, M, K, B, seed = 4, 24, 48, 4, 31
    Ts, nw, nm = [0.5, 0.05], 1, 2
    r = driver.magnetization_curve(L, M, Ts, nw, nm, B, seed=seed, JH=4.0, n_energy=K)
    S = wl.make_spins(L, seed)
    sweep, ok_all = 0, True
    for i, T in enumerate(Ts):
        fn = lambda S_, p, u: oracle.sweep(L, 1.0, 4.0, T, 0.0, M, K, 0, 4.0, S_, 1, B, p, u, nthreads=4)
        ref = rng.run_chain(fn, S, seed, sweep, nw + nm)
        S, sweep = ref["spins"], sweep + nw + nm
        ok_all &= bool((np.abs(-ref["dS"] - np.log(ref["uniforms"])) > 1e-8).all())
        if ok_all:
            assert np.abs(r["series"][i] - ref["magnetization"][nw:]).max() <= 1e-14
            assert abs(r["acceptance"][i] - ref["n_accepted"][nw:].sum() / (nm * L ** 3)) < 1e-15
    assert ok_all and np.abs(r["spins"] - S).max() <= 4e-16
    assert r["acceptance"][0] > r["acceptance"][1]          # hotter chain accepts more


def test_set_temperature_validates_and_changes_only_beta(oracle):
    """T enters only through beta in Delta S (Eq. (14)): moments unchanged, Delta S equal to the oracle's at the new T."""
    L, M, K = 4, 32, 64
    S = wl.make_spins(L, seed=2)
    sites = np.arange(0, 64, 7, dtype=np.int32)
    props = wl.make_spins(L, seed=3)[sites]
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.05, n_energy=K, max_batch_sites=len(sites))
    g.gfmc_set_spins(ctx, S)
    mu0 = g.gfmc_moments(ctx, sites)
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(g.GfmcError):
            g.gfmc_set_temperature(ctx, bad)
    g.gfmc_set_temperature(ctx, 0.4)
    assert np.array_equal(g.gfmc_moments(ctx, sites), mu0)
    dS = g.gfmc_delta_S(ctx, sites, props)
    ref = np.array([oracle.site_dS(L, 1.0, 4.0, 0.4, 0.0, M, K, 0, 4.0, S, int(s), props[i]) for i, s in enumerate(sites)])
    assert (np.abs(dS - ref) / np.maximum(1.0, np.abs(ref))).max() <= 1e-9
    g.gfmc_destroy(ctx)


def test_parallel_chains_equal_serial_chains():
    """driver.magnetization_curve_parallel: every temperature is an independent chain on its own context/stream/thread
    (the paper's MPI level, on one GPU); each must equal the same chain run alone, bit for bit."""
    from paper_1303_6016_b200 import driver
    L, M, B, seed = 4, 32, 1, 21
    Ts = [0.4, 0.2, 0.1, 0.05, 0.3, 0.15, 0.08, 0.03, 0.25, 0.12]
    r = driver.magnetization_curve_parallel(L, M, Ts, 2, 3, B, seed=seed, JH=4.0, n_energy=64)
    assert r["T"] == Ts
    S0 = wl.make_spins(L, seed)
    for i in (0, 3, 9):
        ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=Ts[i], n_energy=64, max_batch_sites=B)
        g.gfmc_set_spins(ctx, S0)
        g.gfmc_run(ctx, seed + i, 0, 2, B)
        mag, nacc = g.gfmc_run(ctx, seed + i, 2, 3, B)
        assert np.array_equal(mag, r["series"][i]) and np.array_equal(g.gfmc_get_spins(ctx), r["spins"][i])
        g.gfmc_destroy(ctx)


def test_graph_replay_equals_individual_launches():
    """Sweeps on small lattices replay one CUDA graph per batch (device-side batch cursor); flags = GFMC_FLAG_NO_GRAPH launches every
    kernel individually.  Same chain bit for bit, incl. a ragged last batch (32 sites per colour in batches of 5) and both models."""
    for model, JH in ((g.GFMC_MODEL_HUND, 4.0), (g.GFMC_MODEL_DEX_INF, 0.0)):
        res = {}
        for flag in ("1", "0"):
            ctx = g.gfmc_create(L=4, M=24, t=1.0, JH=JH, T=0.1, n_energy=64, max_batch_sites=5, model=model,
                                flags=g.GFMC_FLAG_NO_GRAPH if flag == "1" else 0)
            g.gfmc_set_spins(ctx, wl.make_spins(4, seed=8))
            mag, nacc = g.gfmc_run(ctx, 3, 0, 3, 5)
            res[flag] = (mag, nacc, g.gfmc_get_spins(ctx), g.gfmc_launch_counts(ctx))
            g.gfmc_destroy(ctx)
        assert np.array_equal(res["0"][0], res["1"][0]) and np.array_equal(res["0"][1], res["1"][1])
        assert np.array_equal(res["0"][2], res["1"][2])
        assert res["0"][3][0] == res["1"][3][0]                    # same number of fused-step launches counted either way


def test_run_summary_is_alg1_lines_16_17(oracle):
    """gfmc_run_summary = M/S of Alg. 1 lines 16-17, accumulated on the device, against numpy on the per-sweep
    series of the same call; refused before any run; reset by every run."""
    L, M, B = 4, 16, 4
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.2, max_batch_sites=B)
    g.gfmc_set_spins(ctx, wl.make_spins(L, seed=6))
    with pytest.raises(g.GfmcError, match="ESTATE"):
        g.gfmc_run_summary(ctx)
    mag, nacc = g.gfmc_run(ctx, 5, 0, 7, B)
    st = g.gfmc_run_summary(ctx)
    assert st["n_sweeps"] == 7
    assert abs(st["mean"] - mag.mean()) <= 1e-15
    assert abs(st["stderr"] - mag.std(ddof=1) / np.sqrt(7)) <= 1e-15
    assert abs(st["acceptance"] - nacc.sum() / (7 * L ** 3)) <= 1e-15
    mag1, nacc1 = g.gfmc_run(ctx, 5, 7, 1, B)
    st = g.gfmc_run_summary(ctx)
    assert st["n_sweeps"] == 1 and st["mean"] == mag1[0] and np.isnan(st["stderr"]) and st["acceptance"] == nacc1[0] / L ** 3
    g.gfmc_destroy(ctx)


def test_dex_odd_L_refuses_batches_of_neighbours():
    """(x+y+z) mod 2 is a proper colouring only for even L; in the J_H->inf model two neighbouring flips share a bond, so odd L with
    batch_sites > 1 is refused (GFMC_EINVAL) while the sequential algorithm (batch_sites = 1) runs on any lattice."""
    L, M = 5, 8
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=0.0, T=0.1, max_batch_sites=8, model=g.GFMC_MODEL_DEX_INF)
    S = wl.make_spins(L, seed=3)
    g.gfmc_set_spins(ctx, S)
    with pytest.raises(g.GfmcError, match="odd L"):
        g.gfmc_run(ctx, 1, 0, 1, 8)
    with pytest.raises(g.GfmcError, match="odd L"):
        g.gfmc_sweep(ctx, 1, 2, np.zeros((1, L ** 3, 3)), np.full((1, L ** 3), 0.5))
    assert np.array_equal(g.gfmc_get_spins(ctx), S)
    mag, nacc = g.gfmc_run(ctx, 1, 0, 1, 1)
    assert 0 <= nacc[0] <= L ** 3
    g.gfmc_destroy(ctx)


def test_graph_replayed_sweeps_with_device_pointers_equal_host_sweeps():
    """Several graph-replayed sweeps in one call with device-resident trial moves and logs (staged through the context's own
    buffers so that one graph per batch size serves every sweep) == the same call with host arrays."""
    import torch
    L, M, B, ns = 6, 16, 5, 3
    cfg = wl.Config(0, L, 1.0, 4.0, 0.1, 0.0, "sphere", 0.0, 12, M, 2 * M, B, ns)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=B)
    g.gfmc_set_spins(ctx, S)
    out_h = g.gfmc_sweep(ctx, ns, B, prop, uni)
    S_h = g.gfmc_get_spins(ctx)
    g.gfmc_set_spins(ctx, S)
    out_d = g.gfmc_sweep(ctx, ns, B, torch.from_numpy(prop).cuda(), torch.from_numpy(uni).cuda())
    for k in out_h:
        assert np.array_equal(out_d[k].cpu().numpy(), out_h[k]), k
    assert np.array_equal(g.gfmc_get_spins(ctx), S_h)
    g.gfmc_destroy(ctx)


def test_step_loop_timing_is_bounded_in_long_sweeps():
    """A sequential sweep on the streaming path has thousands of batches; only the first 64 are timed (bounded event pool) and
    n_steps counts exactly those, so ms / n_steps stays the average fused-step duration."""
    L, M = 14, 4
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=8)
    g.gfmc_set_spins(ctx, wl.make_spins(L, seed=4))
    g.gfmc_run(ctx, 2, 0, 1, 8)                       # 2 x 172 batches
    ms, steps = g.gfmc_last_step_loop_ms(ctx)
    assert steps == 64 * (M // 2) and ms > 0.0
    assert g.gfmc_launch_counts(ctx)[0] == 2 * 172 * (M // 2)
    g.gfmc_destroy(ctx)
