"""One Monte Carlo chain whose frozen batches are sharded over G GPUs -- SURVEY.md §8(e).

The start vectors of a batch are independent, so a batch's site list is cut into G contiguous shares (kept even-sized where a
work-buffer slot holds two sites); every rank holds the whole spin field (24 B x N, replicated) and its own gfmc context, runs
rows a2-a6 and the accept test for ITS share (`gfmc_decide_batch`: the configuration is not modified), the ranks exchange
(accepted, dS) with ONE all-gather per batch (<= 9 bytes per site), and every rank applies ALL accepted flips
(`gfmc_apply_flips`).  No halo exchange: each rank holds whole vectors.  The paper's own, coarser level -- independent chains per
rank, PAPER.md:259-263 -- is what `bench.py --gpus N` runs by default.

Orchestration only: every number comes from libgfmc.so; the collective is torch.distributed's (NCCL for CUDA tensors -- one
process per GPU -- or gloo for host tensors, which is what the tests use).  Decisions do not depend on how a batch is cut, so the
sharded chain has the same accept flags and spins, bit for bit, as the single-GPU chain (tests/test_sharded_host.py on CPU, tests/test_gpu_sharded.py on one GPU).
"""
from __future__ import annotations

import numpy as np

from . import binding as g
from . import workload as wl


def shard_bounds(n: int, world: int, align: int = 1):
    """Contiguous, balanced cut of a list of n sites into `world` shares whose sizes are multiples of `align` (except the last
    non-empty one): list of (lo, hi) per rank; shares may be empty when n < world * align."""
    units = -(-n // align)                      # shares are counted in units of `align` sites
    out, lo = [], 0
    for r in range(world):
        cnt = units // world + (1 if r < units % world else 0)
        hi = min(n, lo + cnt * align)
        out.append((lo, hi))
        lo = hi
    return out


def gather_decisions(dS_loc: np.ndarray, acc_loc: np.ndarray, bounds, rank: int, group=None, device=None):
    """The one exchange step of a sharded batch: all-gather of every rank's (dS, accepted).  Shares are padded to the largest one
    (all_gather wants equal sizes) and cut back with `bounds`.  Returns (dS[n], accepted[n] uint8) of the whole batch."""
    import torch
    import torch.distributed as dist
    world = len(bounds)
    n = bounds[-1][1]
    if world == 1:
        return dS_loc, acc_loc
    width = max(hi - lo for lo, hi in bounds)
    dev = device if device is not None else "cpu"
    # one buffer per rank: dS as float64 followed by the flags widened to float64 (one collective instead of two)
    mine = torch.zeros(2 * width, dtype=torch.float64, device=dev)
    lo, hi = bounds[rank]
    mine[: hi - lo] = torch.as_tensor(np.ascontiguousarray(dS_loc), dtype=torch.float64).to(dev)
    mine[width: width + hi - lo] = torch.as_tensor(np.ascontiguousarray(acc_loc).astype(np.float64)).to(dev)
    allbuf = torch.empty(world * 2 * width, dtype=torch.float64, device=dev)
    dist.all_gather_into_tensor(allbuf, mine, group=group)
    allbuf = allbuf.cpu().numpy().reshape(world, 2, width)
    dS = np.empty(n, dtype=np.float64)
    acc = np.empty(n, dtype=np.uint8)
    for r, (lo, hi) in enumerate(bounds):
        dS[lo:hi] = allbuf[r, 0, : hi - lo]
        acc[lo:hi] = allbuf[r, 1, : hi - lo].astype(np.uint8)
    return dS, acc


_gather_buffers = {}       # (device, world, width) -> (mine, allbuf): reused from batch to batch


def gather_decisions_device(dS_loc, acc_loc, bounds, rank: int, group=None):
    """gather_decisions for CUDA tensors: the (dS, accepted) of this rank's share go from the buffers gfmc_decide_batch wrote into
    one preallocated send buffer, ONE all-gather (NCCL: device to device over NVLink; gloo, which the one-GPU tests use: staged
    through the host), and come back as device tensors (dS[n] float64, accepted[n] uint8) that gfmc_apply_flips reads."""
    import torch
    import torch.distributed as dist
    world = len(bounds)
    if world == 1:
        return dS_loc, acc_loc
    width = max(hi - lo for lo, hi in bounds)
    dev = dS_loc.device
    key = (dev, world, width)
    if key not in _gather_buffers:
        _gather_buffers[key] = (torch.zeros(2 * width, dtype=torch.float64, device=dev),
                                torch.empty(world * 2 * width, dtype=torch.float64, device=dev))
    mine, allbuf = _gather_buffers[key]
    lo, hi = bounds[rank]
    mine[: hi - lo] = dS_loc
    mine[width: width + hi - lo] = acc_loc.to(torch.float64)
    if dist.get_backend(group) == "nccl":
        dist.all_gather_into_tensor(allbuf, mine, group=group)
    else:
        host = torch.empty(world * 2 * width, dtype=torch.float64)
        dist.all_gather_into_tensor(host, mine.cpu(), group=group)
        allbuf.copy_(host)
    parts = allbuf.view(world, 2, width)
    dS = torch.cat([parts[r, 0, : hi - lo] for r, (lo, hi) in enumerate(bounds)])
    acc = torch.cat([parts[r, 1, : hi - lo] for r, (lo, hi) in enumerate(bounds)]).to(torch.uint8)
    return dS, acc


def sharded_update_batch(ctx, sites, proposals, uniforms, rank: int, world: int, group=None, device=None):
    """gfmc_update_batch for a batch sharded over `world` ranks (call on every rank with the same arguments).
    Returns (dS[n], accepted[n]) of the WHOLE batch; afterwards every rank's context holds the same configuration.
    Host (numpy) arguments are staged through the host as before; contiguous CUDA tensors stay on the device end to end
    (decide on slices of them, all-gather into a reused device buffer, apply from it).
    `ctx.last_decide_loop_ms` = gfmc_last_step_loop_ms of this rank's gfmc_decide_batch, read BEFORE gfmc_apply_flips (every
    library call resets the step-loop timing when it starts); (0.0, 0) for an empty share."""
    on_device = g._is_torch(sites)
    if not on_device:
        sites = np.ascontiguousarray(sites, dtype=np.int32)
        proposals = np.ascontiguousarray(proposals, dtype=np.float64)
        uniforms = np.ascontiguousarray(uniforms, dtype=np.float64)
    align = 1 if (ctx.params.model == g.GFMC_MODEL_HUND and not ctx.params.ph_symmetry) else 2   # two sites per work-buffer slot
    bounds = shard_bounds(len(sites), world, align)
    lo, hi = bounds[rank]
    ctx.last_decide_loop_ms = (0.0, 0)
    if hi > lo:
        dS_loc, acc_loc = g.gfmc_decide_batch(ctx, sites[lo:hi], proposals[lo:hi], uniforms[lo:hi])
        ctx.last_decide_loop_ms = g.gfmc_last_step_loop_ms(ctx)
    elif on_device:
        import torch
        dS_loc = torch.empty(0, dtype=torch.float64, device=sites.device)
        acc_loc = torch.empty(0, dtype=torch.uint8, device=sites.device)
    else:
        dS_loc, acc_loc = np.empty(0), np.empty(0, dtype=np.uint8)
    if on_device:
        dS, acc = gather_decisions_device(dS_loc, acc_loc, bounds, rank, group)
    else:
        dS, acc = gather_decisions(dS_loc, acc_loc, bounds, rank, group, device)
    g.gfmc_apply_flips(ctx, sites, proposals, acc)
    return dS, acc


def sharded_sweep(ctx, n_sweeps: int, batch_sites: int, proposals, uniforms, rank: int, world: int, group=None, device=None):
    """gfmc_sweep (colour-major frozen batches of `batch_sites`, Algorithm 1) with every batch sharded over the
    ranks: `batch_sites` is the size of the WHOLE batch, each rank's context needs max_batch_sites >= its share.
    proposals [n_sweeps, N, 3], uniforms [n_sweeps, N] indexed by site, identical on all ranks.
    Returns dict(dS, accept, magnetization, n_accepted) like gfmc_sweep."""
    N, L = ctx.N, ctx.L
    dS = np.zeros((n_sweeps, N)); acc = np.zeros((n_sweeps, N), dtype=np.uint8)
    mag = np.zeros(n_sweeps); nacc = np.zeros(n_sweeps, dtype=np.int64)
    colours = [wl.colour_sites(L, 0), wl.colour_sites(L, 1)]
    for s in range(n_sweeps):
        for order in colours:
            for st in range(0, len(order), batch_sites):
                b = order[st:st + batch_sites]
                d, a = sharded_update_batch(ctx, b, proposals[s][b], uniforms[s][b], rank, world, group, device)
                dS[s][b] = d; acc[s][b] = a
        mag[s] = g.gfmc_magnetization(ctx)
        nacc[s] = int(acc[s].sum())
    return dict(dS=dS, accept=acc, magnetization=mag, n_accepted=nacc)
