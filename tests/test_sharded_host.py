"""Host logic of the sharded chain (paper_1303_6016_b200/sharded.py) -- no GPU: the cut of a batch into per-rank
shares and the one all-gather per batch, with world_size 2 over gloo."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import numpy as np

from paper_1303_6016_b200 import sharded

ROOT = Path(__file__).resolve().parent.parent


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_bounds_cover_the_batch_in_order():
    for n in (0, 1, 2, 7, 512, 513, 2048, 4095):
        for world in (1, 2, 3, 8):
            for align in (1, 2):
                b = sharded.shard_bounds(n, world, align)
                assert len(b) == world and b[0][0] == 0 and b[-1][1] == n
                assert all(b[r][1] == b[r + 1][0] for r in range(world - 1))           # contiguous, in order
                sizes = [hi - lo for lo, hi in b]
                assert min(sizes) >= 0 and sum(sizes) == n
                units = -(-n // align)
                assert max(sizes) <= -(-units // world) * align                        # balanced: nobody exceeds the ceiling share
                nonempty = [s_ for s_ in sizes if s_ > 0]
                assert all(s_ % align == 0 for s_ in nonempty[:-1])                    # only the last non-empty share may be ragged


def test_gather_decisions_two_gloo_ranks(tmp_path):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                          "--master-port", str(free_port()), str(ROOT / "tests" / "sharded_worker.py"), "host", str(tmp_path)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    for rank in (0, 1):
        res = json.loads((tmp_path / f"host_rank{rank}.json").read_text())
        assert len(res) == 5 and all(res.values()), res


def test_single_rank_gather_is_identity():
    d, a = np.array([1.0, -2.0]), np.array([0, 1], dtype=np.uint8)
    d2, a2 = sharded.gather_decisions(d, a, sharded.shard_bounds(2, 1), 0)
    assert d2 is d and a2 is a
