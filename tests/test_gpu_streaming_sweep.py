"""GPU parity of gfmc_sweep / gfmc_run on the STREAMING kernel (`-m gpu`): lattices with L >= 13 take the path
sweep_device -> D2D site gather -> run_moments_batch (TMA rings, balanced work list where it applies, bond refresh between
batches in the J_H->inf model) -> site-indexed proposals, which the small-lattice sweep tests (resident kernel) never reach.
Every element of dS, accept, spins, magnetization and n_accepted is compared with the oracle's Algorithm 1
(PAPER.md:266-306), all three modes of the fused step.  Bars as in test_gpu_parity.py."""
import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl

pytestmark = pytest.mark.gpu

DS_RTOL = 1e-9
TIE = 1e-8


def _ds_close(a, b):
    return np.abs(a - b) <= DS_RTOL * np.maximum(1.0, np.abs(b))


def _create(mode, L, M, K, T, JH, B):
    if mode == "dex":
        return g.gfmc_create(L=L, M=M, t=1.0, JH=0.0, T=T, n_energy=K, max_batch_sites=B, model=g.GFMC_MODEL_DEX_INF)
    if mode == "ph2":                 # one start vector per site AND two Chebyshev steps per pass (cheb_step2.cuh; L = 32, M % 4 == 0)
        return g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=T, n_energy=K, max_batch_sites=B, ph_symmetry=1, flags=g.GFMC_FLAG_TWO_STEP)
    return g.gfmc_create(L=L, M=M, t=1.0, JH=JH, T=T, n_energy=K, max_batch_sites=B, ph_symmetry=1 if mode == "ph" else 0)


def _oracle_sweep(oracle, mode, L, M, K, T, JH, S, ns, B, prop, uni):
    if mode == "dex":
        return oracle.dex_sweep(L, 1.0, T, 0.0, M, K, 0, 4.0, S, ns, B, prop, uni, nthreads=16)
    return oracle.sweep(L, 1.0, JH, T, 0.0, M, K, 0, 4.0, S, ns, B, prop, uni, nthreads=16)


def _check(out, S_gpu, ref, uni):
    margin = -ref["dS"] - np.log(uni)
    assert (np.abs(margin) > TIE).all(), "a decision fell inside the tie window; pick another seed"
    assert np.array_equal(out["accept"], ref["accept"])                    # bit-exact decisions
    assert _ds_close(out["dS"], ref["dS"]).all()
    assert np.array_equal(S_gpu, ref["spins"])                             # spins are copies of the proposals
    assert np.array_equal(out["n_accepted"], ref["n_accepted"])
    assert np.abs(out["magnetization"] - ref["magnetization"]).max() < 1e-14


@pytest.mark.parametrize("mode", ["hund", "ph", "dex"])
@pytest.mark.parametrize("L,M,K,B,ns", [
    (16, 32, 64, 512, 2),     # 4 + 4 batches per sweep; 256 / 128 two-pair columns on 148 SMs: the balanced work list is active
    (20, 24, 48, 700, 1),     # run-time-L ring (no compile-time instantiation), plane not a multiple of 32, ragged last batch
])
def test_sweep_streaming_kernel_matches_oracle(oracle, mode, L, M, K, B, ns):
    JH, T = 8.0, 0.05
    if mode == "dex":                 # the J_H->inf oracle recomputes every bond amplitude in every application: keep its share small
        M, K = M // 2, K // 2
    cfg = wl.Config(0, L, 1.0, JH, T, 0.0, "sphere", 0.0, 100 + L, M, K, B, ns)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
    ref = _oracle_sweep(oracle, mode, L, M, K, T, JH, S, ns, B, prop, uni)
    ctx = _create(mode, L, M, K, T, JH, B)
    g.gfmc_set_spins(ctx, S)
    out = g.gfmc_sweep(ctx, ns, B, prop, uni)
    launches = g.gfmc_launch_counts(ctx)[0]
    nb = sum(-(-len(wl.colour_sites(L, c)) // B) for c in (0, 1))
    assert launches == ns * nb * (M // 2)                                  # streaming kernel: one launch per fused step and batch
    S_gpu = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    _check(out, S_gpu, ref, uni)
    assert 0 < out["n_accepted"].sum() < ns * L ** 3


@pytest.mark.parametrize("mode", ["hund", "ph", "dex"])
def test_sweep_streaming_device_pointers_and_logs(oracle, mode):
    """Same path with device-resident proposals / uniforms / logs (mem = GFMC_DEVICE), several sweeps in one call."""
    import torch
    L, M, K, B, ns, JH, T = 16, 16, 32, 1024, 2, 8.0, 0.1
    cfg = wl.Config(0, L, 1.0, JH, T, 0.0, "cone", 0.9, 77, M, K, B, ns)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
    ref = _oracle_sweep(oracle, mode, L, M, K, T, JH, S, ns, B, prop, uni)
    ctx = _create(mode, L, M, K, T, JH, B)
    g.gfmc_set_spins(ctx, S)
    out = g.gfmc_sweep(ctx, ns, B, torch.from_numpy(prop).cuda(), torch.from_numpy(uni).cuda())
    out = {k: v.cpu().numpy() for k, v in out.items()}
    S_gpu = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    _check(out, S_gpu, ref, uni)


@pytest.mark.parametrize("mode", ["hund", "ph", "dex"])
def test_run_streaming_kernel_matches_oracle_chain(oracle, mode):
    """gfmc_run (device-side Philox trial moves) at L = 16 == the oracle's chain fed by the oracle's own generator;
    and bit-identical to its replay through gfmc_sweep."""
    from oracle import rng
    L, M, K, B, JH, T, seed, first, n = 16, (12 if mode == "dex" else 24), (24 if mode == "dex" else 48), 512, 8.0, 0.05, 4242, 7, 2
    S = wl.make_spins(L, seed=61)
    fn = lambda S_, p, u: _oracle_sweep(oracle, mode, L, M, K, T, JH, S_, 1, B, p, u)
    ref = rng.run_chain(fn, S, seed, first, n)
    ctx = _create(mode, L, M, K, T, JH, B)
    g.gfmc_set_spins(ctx, S)
    mag, nacc = g.gfmc_run(ctx, seed, first, n, B)
    S_gpu = g.gfmc_get_spins(ctx)
    g.gfmc_set_spins(ctx, S)
    P = np.stack([g.gfmc_random_proposals(ctx, seed, first + s)[0] for s in range(n)])
    U = np.stack([g.gfmc_random_proposals(ctx, seed, first + s)[1] for s in range(n)])
    r2 = g.gfmc_sweep(ctx, n, B, P, U)
    S_replay = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    assert np.array_equal(S_replay, S_gpu) and np.array_equal(r2["magnetization"], mag) and np.array_equal(r2["n_accepted"], nacc)
    margin = -ref["dS"] - np.log(ref["uniforms"])
    assert (np.abs(margin) > TIE).all(), "a decision fell inside the tie window; pick another seed"
    assert np.array_equal(r2["accept"], ref["accept"])
    assert _ds_close(r2["dS"], ref["dS"]).all()
    assert np.array_equal(nacc, ref["n_accepted"])
    assert np.abs(S_gpu - ref["spins"]).max() <= 4e-16                    # trial spins: sincos vs cos, sin of two libraries
    assert np.abs(mag - ref["magnetization"]).max() <= 1e-14


# --------------------------------------------------------------------------- two Chebyshev steps per pass through the sweep / run drivers
def test_two_step_sweep_matches_oracle(oracle):
    """GFMC_FLAG_TWO_STEP through gfmc_sweep at L = 32: four work buffers rotating across the 47 consecutive batches of a sweep,
    B = 700 (odd number of slots' worth of sites in the ragged last batch of each colour: 16384 = 23 * 700 + 284), site-indexed
    proposals.  Every element against the oracle's Algorithm 1, which knows neither the symmetry shortcut nor the two-step pass."""
    L, M, K, B, JH, T = 32, 16, 32, 700, 8.0, 0.05
    cfg = wl.Config(0, L, 1.0, JH, T, 0.0, "sphere", 0.0, 132, M, K, B, 1)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    ref = _oracle_sweep(oracle, "hund", L, M, K, T, JH, S, 1, B, prop, uni)
    ctx = _create("ph2", L, M, K, T, JH, B)
    g.gfmc_set_spins(ctx, S)
    out = g.gfmc_sweep(ctx, 1, B, prop, uni)
    nb = sum(-(-len(wl.colour_sites(L, c)) // B) for c in (0, 1))
    assert g.gfmc_launch_counts(ctx)[0] == nb * (M // 4)                    # two fused steps per launch
    S_gpu = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    _check(out, S_gpu, ref, uni)
    assert 0 < out["n_accepted"].sum() < L ** 3


def test_two_step_run_matches_oracle_chain(oracle):
    """gfmc_run (device-side Philox trial moves) with GFMC_FLAG_TWO_STEP at L = 32 == the oracle's chain fed by the oracle's own
    generator, and bit-identical to the one-step one-vector kernel's decisions."""
    from oracle import rng
    L, M, K, B, JH, T, seed, first, n = 32, 8, 16, 701, 8.0, 0.05, 99, 3, 1
    S = wl.make_spins(L, seed=62)
    fn = lambda S_, p, u: _oracle_sweep(oracle, "hund", L, M, K, T, JH, S_, 1, B, p, u)
    ref = rng.run_chain(fn, S, seed, first, n)
    res = {}
    for mode in ("ph2", "ph"):
        ctx = _create(mode, L, M, K, T, JH, B)
        g.gfmc_set_spins(ctx, S)
        mag, nacc = g.gfmc_run(ctx, seed, first, n, B)
        res[mode] = (mag, nacc, g.gfmc_get_spins(ctx))
        g.gfmc_destroy(ctx)
    mag, nacc, S_gpu = res["ph2"]
    margin = -ref["dS"] - np.log(ref["uniforms"])
    assert (np.abs(margin) > TIE).all(), "a decision fell inside the tie window; pick another seed"
    assert np.array_equal(nacc, ref["n_accepted"])
    assert np.abs(S_gpu - ref["spins"]).max() <= 4e-16
    assert np.abs(mag - ref["magnetization"]).max() <= 1e-14
    assert np.array_equal(S_gpu, res["ph"][2]) and np.array_equal(nacc, res["ph"][1])
