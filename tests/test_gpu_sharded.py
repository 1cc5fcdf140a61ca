"""SURVEY.md §8(e) on hardware that has one GPU: two ranks (two processes, gloo for the exchange, both on cuda:0 -- their kernels
never wait on each other, only the hosts do) run ONE chain whose frozen batches are cut in two; the result must be the
single-rank chain: accept flags and spins bit for bit, Delta S to rounding (`-m gpu`)."""
import json
import os
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

import paper_1303_6016_b200 as g
from paper_1303_6016_b200 import workload as wl
from tests.test_sharded_host import free_port

pytestmark = pytest.mark.gpu

ROOT = Path(__file__).resolve().parent.parent

CASES = {
    "hund": dict(L=16, M=16, K=32, B=512, ns=1, JH=8.0, T=0.05, seed=71, kw={}),
    "ph": dict(L=16, M=16, K=32, B=301, ns=1, JH=8.0, T=0.05, seed=72, kw=dict(ph_symmetry=1)),       # odd batch: ragged last share
    "dex": dict(L=16, M=12, K=24, B=512, ns=1, JH=0.0, T=0.05, seed=73, kw=dict(model=1)),           # bond refresh after every batch
    "ph2": dict(L=32, M=8, K=16, B=701, ns=1, JH=8.0, T=0.05, seed=75, kw=dict(ph_symmetry=1, flags=8)),   # GFMC_FLAG_TWO_STEP: two steps per pass, odd shares
    "small": dict(L=6, M=16, K=32, B=20, ns=2, JH=4.0, T=0.1, seed=74, kw={}),                       # resident kernel, two sweeps
}


def test_two_rank_sharded_chain_equals_single_rank_chain(tmp_path):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                          "--master-port", str(free_port()), str(ROOT / "tests" / "sharded_worker.py"), "gpu", str(tmp_path), json.dumps(CASES)],
                         capture_output=True, text=True, env=env, timeout=1200)
    assert out.returncode == 0, out.stderr[-3000:]
    for name, c in CASES.items():
        L, M, K, B, ns = c["L"], c["M"], c["K"], c["B"], c["ns"]
        cfg = wl.Config(0, L, 1.0, c["JH"], c["T"], 0.0, "sphere", 0.0, c["seed"], M, K, B, ns)
        S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
        ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=c["JH"], T=c["T"], n_energy=K, max_batch_sites=B, **c["kw"])
        g.gfmc_set_spins(ctx, S)
        ref = g.gfmc_sweep(ctx, ns, B, prop, uni)
        S_ref = g.gfmc_get_spins(ctx)
        g.gfmc_destroy(ctx)
        for rank in (0, 1):
            r = np.load(tmp_path / f"gpu_{name}_rank{rank}.npz")
            assert np.array_equal(r["accept"], ref["accept"]), (name, rank)
            assert np.array_equal(r["spins"], S_ref), (name, rank)                       # every replica holds the same configuration
            assert np.array_equal(r["n_accepted"], ref["n_accepted"])
            assert np.abs(r["dS"] - ref["dS"]).max() <= 1e-11 * max(1.0, np.abs(ref["dS"]).max()), name
            assert np.abs(r["magnetization"] - ref["magnetization"]).max() < 1e-14
        assert 0 < ref["n_accepted"].sum() < ns * L ** 3


def test_decide_batch_leaves_the_configuration_alone_and_apply_flips_chunks():
    L, M = 6, 16
    S = wl.make_spins(L, seed=5)
    sites = wl.colour_sites(L, 0)[:40]
    prop = wl.make_spins(L, seed=6)[sites]
    uni = np.full(len(sites), 0.3)
    ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=64)
    g.gfmc_set_spins(ctx, S)
    dS, acc = g.gfmc_decide_batch(ctx, sites, prop, uni)
    assert np.array_equal(g.gfmc_get_spins(ctx), S)                                       # nothing applied
    dS2, acc2 = g.gfmc_update_batch(ctx, sites, prop, uni)
    assert np.array_equal(dS, dS2) and np.array_equal(acc, acc2)
    S_upd = g.gfmc_get_spins(ctx)
    g.gfmc_destroy(ctx)
    small = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=7)               # apply_flips stages the list in chunks of 7
    g.gfmc_set_spins(small, S)
    g.gfmc_apply_flips(small, sites, prop, acc)
    assert np.array_equal(g.gfmc_get_spins(small), S_upd)
    with pytest.raises(g.GfmcError, match="out of range"):
        g.gfmc_apply_flips(small, np.array([L ** 3], dtype=np.int32), prop[:1], acc[:1])
    with pytest.raises(g.GfmcError, match="gfmc_apply_flips: sites must be distinct"):       # a wrong shard cut repeats a site
        g.gfmc_apply_flips(small, np.array([3, 5, 3], dtype=np.int32), prop[:3], acc[:3])
    with pytest.raises(g.GfmcError, match="gfmc_decide_batch: n_sites 8 > max_batch_sites 7"):  # errors name the entry point that was called
        g.gfmc_decide_batch(small, sites[:8], prop[:8], uni[:8])
    assert np.array_equal(g.gfmc_get_spins(small), S_upd)
    g.gfmc_destroy(small)
    ex = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.1, max_batch_sites=8, exact_batch_sites=8)
    g.gfmc_set_spins(ex, S)
    g.gfmc_set_batch_mode(ex, g.GFMC_BATCH_EXACT)
    with pytest.raises(g.GfmcError, match="FROZEN"):
        g.gfmc_decide_batch(ex, sites[:4], prop[:4], uni[:4])
    g.gfmc_destroy(ex)


def test_bench_shard_two_ranks_one_gpu_prints_the_contract_line():
    """`bench.py --gpus 2 --shard` end to end (round-2 finding: it divided by zero after the timed run because gfmc_apply_flips resets
    the step-loop timing): the command starts its own two ranks, both on cuda:0 with gloo for the exchange, device-resident value leg
    and host-buffer e2e leg, and rank 0 prints the JSON line."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--shard", "--dist-backend", "gloo", "--config", "3",
                          "--steps", "2", "--warmup", "1", "--no-cpu", "--no-modes"], capture_output=True, text=True, timeout=1200, env=env)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["scaling"] == "strong" and line["config"]["replicas"] == 1
    assert np.isfinite(line["roofline"]["frac"]) and 0.0 < line["roofline"]["frac"] < 1.5
    assert line["roofline"]["launches_timed"] == 2 * 256 and line["value"] > 0 and line["e2e"]["value"] > 0
