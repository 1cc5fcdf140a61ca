"""Host-side checks of bench.py: the max-over-ranks / sum-of-units aggregation used for N > 1 replicas is
exercised with world_size 2 over gloo on CPU; the reference arm's JSON contract is checked on a tiny config."""
import json
import os
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
t, u = bench.aggregate_over_ranks(1.0 + rank, 10.0 * (rank + 1), dist.get_world_size())
dist.barrier()
if rank == 0:
    print(json.dumps({{"t": t, "u": u}}))
dist.destroy_process_group()
"""


def test_aggregate_over_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=str(ROOT)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29731", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    res = json.loads(line)
    assert res["t"] == 2.0 and res["u"] == 30.0            # MAX of times, SUM of units


def test_single_rank_aggregate_is_identity():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.aggregate_over_ranks(1.5, 7.0, 1) == (1.5, 7.0)


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "H-applications/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["dtype"] == "f64" and line["vs_baseline"] is None


def test_gpus_flag_spawns_its_own_ranks():
    """`python bench.py --gpus 2 ...` without torchrun must start two ranks itself (round-2 finding: it used to run one replica and
    print n_gpus 1).  The reference arm needs no GPU: rank 0 prints the line, rank 1 exits 0 without work."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "1", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # one line, from rank 0
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["world_size"] == 2 and line["impl"] == "reference"
