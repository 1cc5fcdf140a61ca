"""Worker of tests/test_sharded_host.py and tests/test_gpu_sharded.py (launched by torch.distributed.run, gloo backend).

mode "host": no GPU, no library -- every rank fabricates the decisions of ITS share from a deterministic function of the site and
the ranks exchange them with paper_1303_6016_b200.sharded.gather_decisions (the one collective of a sharded batch).
mode "gpu": every rank creates its own gfmc context on cuda:0 and runs sharded_sweep; rank 0 writes the result."""
import json
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

import torch.distributed as dist  # noqa: E402

from paper_1303_6016_b200 import sharded, workload as wl  # noqa: E402


def fake_decisions(sites):
    dS = np.sin(sites.astype(np.float64)) * 3.0
    return dS, (dS < 0.5).astype(np.uint8)


def main():
    mode, out = sys.argv[1], Path(sys.argv[2])
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    if mode == "host":
        res = {}
        for n, align in ((1000, 1), (7, 2), (1, 1), (513, 2), (2, 2)):
            sites = (np.arange(n) * 7 + 3).astype(np.int32)
            bounds = sharded.shard_bounds(n, world, align)
            lo, hi = bounds[rank]
            d, a = fake_decisions(sites[lo:hi])
            dS, acc = sharded.gather_decisions(d, a, bounds, rank)
            ref_d, ref_a = fake_decisions(sites)
            res[f"{n}/{align}"] = bool(np.array_equal(dS, ref_d) and np.array_equal(acc, ref_a))
        dist.barrier()
        (out / f"host_rank{rank}.json").write_text(json.dumps(res))
    else:
        import paper_1303_6016_b200 as g
        cfgs = json.loads(sys.argv[3])
        for name, c in cfgs.items():
            L, M, K, B, ns = c["L"], c["M"], c["K"], c["B"], c["ns"]
            cfg = wl.Config(0, L, 1.0, c["JH"], c["T"], 0.0, "sphere", 0.0, c["seed"], M, K, B, ns)
            S, prop, uni = wl.make_workload(cfg, n_sweeps=ns)
            share = -(-B // world) + 1
            ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=c["JH"], T=c["T"], n_energy=K, max_batch_sites=share, **c["kw"])
            g.gfmc_set_spins(ctx, S)
            r = sharded.sharded_sweep(ctx, ns, B, prop, uni, rank, world)
            S_end = g.gfmc_get_spins(ctx)
            g.gfmc_destroy(ctx)
            np.savez(out / f"gpu_{name}_rank{rank}.npz", spins=S_end, **r)
        dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
