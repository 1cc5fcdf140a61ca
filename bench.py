#!/usr/bin/env python
"""bench.py -- throughput of the GFMC hot path on B200.

A "step" is one pass of the whole hot path over one batch of synthetic input:
one frozen-batch Metropolis update (`gfmc_update_batch`) of a 2048-site checkerboard batch of BASELINE.json's
config 4 (L=32, t=1, J_H=8, T=0.02, M=1024, K=2048; 4096 start vectors, M/2 = 512 fused Chebyshev steps, Green's
functions, Delta S_eff, accept, spin update) followed by the magnetization.  `value` is Chebyshev
H-applications/s (start vectors x fused steps per second) over the WHOLE step with inputs resident in HBM;
`e2e` is the same metric through the C ABI with host buffers.  N > 1 runs N independent replicas (the paper's
own outer level: independent Monte Carlo chains per rank) -- no data-path collective.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "Chebyshev H-applications/s (vectors*steps/s) over whole GFMC batch updates at L=32"      # config 4, the headline


def metric_name(cfg):
    return METRIC if cfg.L == 32 else METRIC.replace("L=32", f"L={cfg.L}")
UNIT = "H-applications/s"


# ----------------------------------------------------------------------------- helpers
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def aggregate_over_ranks(elapsed_s: float, units: float, world: int):
    """Barrier-bracketed timing contract: time = MAX over ranks, units = SUM over ranks.
    Uses torch.distributed when world > 1 (nccl on GPUs, gloo in the CPU tests)."""
    if world == 1:
        return elapsed_s, units
    import torch
    import torch.distributed as dist
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    t = torch.tensor([elapsed_s], dtype=torch.float64, device=dev)
    u = torch.tensor([units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        return float(json.loads(f.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def sustained_copy_gbs(dev, seconds=1.5):
    """Context for the roofline fraction: the same STREAM-style copy MEASURED_PEAKS.json's `hbm_gbs` comes from (torch b.copy_(a), read + write
    bytes), but back to back for `seconds` instead of best-of-10 bursts -- what plain copying sustains under the 1000 W cap on THIS box, next
    to which a kernel timed inside a long step loop should be read.  Not the denominator of `frac` (that stays the measured burst peak)."""
    import torch
    n = 1 << 29                                                # 2 x 1 GiB of bf16
    a = torch.empty(n, dtype=torch.bfloat16, device=dev).fill_(1.0)
    b = torch.empty_like(a)
    for _ in range(3):
        b.copy_(a)
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 0
    t0 = time.perf_counter()
    e0.record()
    while time.perf_counter() - t0 < seconds:
        for _ in range(20):
            b.copy_(a)
        reps += 20
        torch.cuda.synchronize(dev)
    e1.record()
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1)
    del a, b
    return 2.0 * n * 2 * reps / (ms * 1e-3) / 1e9


def ncu_traffic():
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the fused step kernel, from the committed
    summary of the `ncu --set full` capture: profiles/step_kernel_traffic.csv (the command is in the .md beside it)."""
    f = ROOT / "profiles" / "step_kernel_traffic.csv"
    try:
        import csv
        rows = list(csv.reader(f.read_text().strip().splitlines()))      # the kernel name holds a comma inside quotes
        return float(rows[1][rows[0].index("dram_bytes_per_launch")])
    except Exception:
        return None


# ----------------------------------------------------------------------------- CPU oracle legs
def oracle_rate(cfg, target_s: float, nthreads: int):
    """Times the oracle's plain three-term recursion (Eq. 26, no doubling) AS IT STANDS on the host cores, on a
    bounded sample: `2*nthreads` start sites of the config's lattice, M_s moments each (M_s - 1 H-applications per
    start vector, two start vectors per site).  Returns (H-applications/s, description)."""
    from oracle import oracle
    from paper_1303_6016_b200 import workload as wl
    S, _, _ = wl.make_workload(cfg, n_sweeps=1)
    n_sites = max(2 * nthreads, 16)
    sites = wl.colour_sites(cfg.L, 0)[:n_sites]
    t0 = time.perf_counter()
    oracle.moments_many(cfg.L, cfg.t, cfg.JH, S, sites, 5, nthreads=nthreads)       # calibration: 4 applications
    dt = max(time.perf_counter() - t0, 1e-4)
    rate0 = n_sites * 2 * 4 / dt
    Ms = int(max(9, target_s * rate0 / (2 * n_sites) + 1))
    if Ms > cfg.M:                                   # full-length recursions: take more start sites instead
        n_sites = int(min(len(wl.colour_sites(cfg.L, 0)), max(n_sites, n_sites * Ms // cfg.M // nthreads * nthreads)))
        sites = wl.colour_sites(cfg.L, 0)[:n_sites]
        Ms = cfg.M
    t0 = time.perf_counter()
    oracle.moments_many(cfg.L, cfg.t, cfg.JH, S, sites, Ms, nthreads=nthreads)
    dt = time.perf_counter() - t0
    happs = n_sites * 2 * (Ms - 1)
    return happs / dt, f"{n_sites} start sites x 2 vectors x {Ms - 1} H-applications of config {cfg.index} (L={cfg.L}), {dt:.1f} s"


def run_reference(args, cfg):
    rank, _, world = dist_env()
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    # a "step" of this arm is a bounded sample of the workload: sized so that the whole run ends within a few minutes
    per_step_s = max(0.5, min(8.0, 150.0 / max(1, args.steps)))
    vals, walls = [], []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        v, desc = oracle_rate(cfg, per_step_s if i >= args.warmup else 1.0, cores)
        if i >= args.warmup:
            vals.append(v); walls.append(time.perf_counter() - t0)
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": metric_name(cfg), "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": float(np.mean(walls)) * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {cfg.index}: L={cfg.L} t={cfg.t} J_H={cfg.JH} T={cfg.T} M={cfg.M}; oracle = plain "
                                   "three-term recursion (no doubling) on a bounded sample per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "world_size": world}       # ranks started (only rank 0 works and prints)
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- further modes (reported beside the headline)
def quick_mode_rate(cfg, B, dev_index, steps, warmup, **mode_kw):
    """Same step (gfmc_update_batch + gfmc_magnetization, device-resident inputs, CUDA events) in another mode of the fused
    kernel: ph_symmetry=1 (Eq. (1), one start vector per site) or model=GFMC_MODEL_DEX_INF (Eq. (2)-(3), the paper's own
    Hamiltonian).  Returns site updates/s, H-applications/s and the step kernel's achieved algorithmic GB/s."""
    import torch
    import paper_1303_6016_b200 as g
    from paper_1303_6016_b200 import workload as wl
    dev = torch.device("cuda", dev_index)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[:B]
    ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=cfg.JH, T=cfg.T, mu=cfg.mu, n_energy=cfg.K, max_batch_sites=B,
                        device=dev_index, **mode_kw)
    g.gfmc_set_spins(ctx, S)
    d_s, d_p, d_u = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (sites, prop[0][sites], uni[0][sites]))
    loop_ms, loop_steps = 0.0, 0
    for i in range(warmup):
        g.gfmc_update_batch(ctx, d_s, d_p, d_u)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(steps):
        g.gfmc_update_batch(ctx, d_s, d_p, d_u)
        ms, n = g.gfmc_last_step_loop_ms(ctx)
        nvec, step_bytes = g.gfmc_last_step_loop_vectors(ctx)
        loop_ms += ms; loop_steps += n
        g.gfmc_magnetization(ctx)
    e1.record()
    torch.cuda.synchronize()
    elapsed = e0.elapsed_time(e1) * 1e-3
    g.gfmc_destroy(ctx)
    avg_launch_s = loop_ms * 1e-3 / max(loop_steps, 1)
    peak, _ = measured_peak()
    return {"site_updates_per_s": B * steps / elapsed, "h_applications_per_s": nvec * (cfg.M // 2) * steps / elapsed,
            "start_vectors_per_batch": nvec, "ms_per_step": elapsed / steps * 1e3, "avg_launch_ms": avg_launch_s * 1e3,
            "algorithmic_bytes_per_launch": step_bytes, "achieved_gbs": step_bytes / avg_launch_s / 1e9,
            "frac": step_bytes / avg_launch_s / 1e9 / peak, "steps": steps, "warmup": warmup}


def config_leg(index, dev_index, steps, warmup):
    """A second, smaller workload of BASELINE.json's `configs` timed in the same driver run (the same step: gfmc_update_batch +
    gfmc_magnetization on device-resident inputs, headline mode), with the roofline of the kernel that serves it: the streaming
    step kernel against the measured HBM rate (L >= 13) or the shared-memory-resident kernel against the shared-memory pipe
    (L <= 12; 36 x 16 B accesses per site and fused step against 128 B/clk per SM at the clock sampled during this leg)."""
    import torch
    from paper_1303_6016_b200 import workload as wl
    cfg = wl.CONFIGS[index]
    sampler = ClockSampler(dev_index)
    sampler.start()
    r = quick_mode_rate(cfg, cfg.batch_sites, dev_index, steps, warmup)
    clocks = sampler.stop()
    out = {"workload": f"config {index}: L={cfg.L} M={cfg.M} K={cfg.K}, {cfg.batch_sites}-site batch ({r['start_vectors_per_batch']} start vectors) per step",
           "site_updates_per_s": r["site_updates_per_s"], "h_applications_per_s": r["h_applications_per_s"], "ms_per_step": r["ms_per_step"],
           "steps": steps, "warmup": warmup, "clocks": clocks}
    if cfg.L <= 12:
        nsm = torch.cuda.get_device_properties(dev_index).multi_processor_count
        smem_bytes = 36.0 * 16.0 * cfg.L ** 3 * cfg.batch_sites * (cfg.M // 2)            # per batch = per launch
        launch_s = r["avg_launch_ms"] * 1e-3 * (cfg.M // 2)                               # avg_launch_ms is per fused STEP
        peak = nsm * 128.0 * (clocks.get("sm_mhz") or 1965.0) * 1e6 / 1e9
        out["roofline"] = {"bound": "smem", "kernel": "cheb_resident_kernel", "achieved": smem_bytes / launch_s / 1e9, "peak": peak, "unit": "GB/s",
                           "frac": smem_bytes / launch_s / 1e9 / peak, "peak_source": "derived: 128 B/clk/SM x SMs x SM clock sampled during this leg",
                           "traffic": None, "algorithmic_bytes_per_launch": smem_bytes, "avg_launch_ms": launch_s * 1e3}
    else:
        peak, src = measured_peak()
        out["roofline"] = {"bound": "hbm", "kernel": "cheb_step_kernel", "achieved": r["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": r["frac"],
                           "peak_source": src, "traffic": None, "algorithmic_bytes_per_launch": r["algorithmic_bytes_per_launch"],
                           "avg_launch_ms": r["avg_launch_ms"]}
    return out


def exact_batch_rate(cfg, Bx, dev_index, steps, warmup):
    """the same lattice / M / K, batches of Bx sites decided sequentially and exactly inside the batch
    (GFMC_BATCH_EXACT: M-1 fused steps with cross-moment read-outs, Bx^2 Green blocks, Woodbury updates), next to the frozen batch of
    the same size.  Returns site updates/s of both."""
    import torch
    import paper_1303_6016_b200 as g
    from paper_1303_6016_b200 import workload as wl
    dev = torch.device("cuda", dev_index)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    sites = wl.colour_sites(cfg.L, 0)[:Bx]
    ctx = g.gfmc_create(L=cfg.L, M=cfg.M, t=cfg.t, JH=cfg.JH, T=cfg.T, mu=cfg.mu, n_energy=cfg.K, max_batch_sites=Bx,
                        exact_batch_sites=Bx, device=dev_index)
    d_s, d_p, d_u = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (sites, prop[0][sites], uni[0][sites]))
    out = {}
    for name, mode in (("frozen", g.GFMC_BATCH_FROZEN), ("exact", g.GFMC_BATCH_EXACT)):
        g.gfmc_set_batch_mode(ctx, mode)
        g.gfmc_set_spins(ctx, S)
        for _ in range(warmup):
            g.gfmc_update_batch(ctx, d_s, d_p, d_u)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            g.gfmc_update_batch(ctx, d_s, d_p, d_u)
        e1.record()
        torch.cuda.synchronize()
        out[name + "_site_updates_per_s"] = Bx * steps / (e0.elapsed_time(e1) * 1e-3)
    # the paper's strictly sequential schedule on the same lattice: one site per batch (frozen and exact coincide)
    g.gfmc_set_batch_mode(ctx, g.GFMC_BATCH_FROZEN)
    g.gfmc_update_batch(ctx, d_s[:1], d_p[:1], d_u[:1])
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for j in range(4):
        g.gfmc_update_batch(ctx, d_s[j:j + 1], d_p[j:j + 1], d_u[j:j + 1])
    e1.record()
    torch.cuda.synchronize()
    out["sequential_site_updates_per_s"] = 4 / (e0.elapsed_time(e1) * 1e-3)
    g.gfmc_destroy(ctx)
    out.update(batch_sites=Bx, steps=steps, warmup=warmup,
               note=f"batches of {Bx} sites at the same lattice/M/K: frozen = M/2 fused steps with doubling; exact = M-1 steps with cross read-outs, "
                    f"{Bx}^2 Green blocks and per-site Woodbury updates; small batches are launch-bound on 148 SMs")
    return out


# ----------------------------------------------------------------------------- CUDA arm
def run_gfmc(args, cfg):
    import torch
    import paper_1303_6016_b200 as g
    from paper_1303_6016_b200 import workload as wl

    rank, local_rank, world = dist_env()
    if world > 1:
        import torch.distributed as dist
        if args.dist_backend == "nccl":
            torch.cuda.set_device(local_rank)
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        else:       # gloo: host-staged exchange; ranks may share a GPU (the one-GPU test of the sharded harness: their kernels never wait on each other)
            dist.init_process_group("gloo")
    dev_index = (local_rank % torch.cuda.device_count()) if world > 1 else 0
    torch.cuda.set_device(dev_index)
    dev = torch.device("cuda", dev_index)

    B, M, K, L = cfg.batch_sites, cfg.M, cfg.K, cfg.L
    if args.batch:
        B = args.batch
    # each rank is an independent replica (its own chain): seed offset by rank
    import dataclasses
    rcfg = dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)
    S, prop, uni = wl.make_workload(rcfg, n_sweeps=1)
    colours = [wl.colour_sites(L, 0), wl.colour_sites(L, 1)]
    batches = [c[i:i + B] for c in colours for i in range(0, len(c), B)]
    shard = bool(args.shard) and world > 1
    if shard:
        # ONE chain, every batch cut into `world` shares (strong scaling); all ranks see the same inputs
        from paper_1303_6016_b200 import sharded
        S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    # the headline arm (--mode hund2) propagates BOTH start vectors of every site (rows a2-a3 as the scope table defines them);
    # --mode ph / dex time another mode of the fused kernel as the main arm (profiling runs; not the headline)
    mode_kw = {"hund2": {}, "ph": dict(ph_symmetry=1), "ph2": dict(ph_symmetry=1, flags=g.GFMC_FLAG_TWO_STEP),
               "dex": dict(model=g.GFMC_MODEL_DEX_INF)}[args.mode]
    if args.ring:                       # diagnostic: ring depths of the streaming kernel (R_cur, R_prev), e.g. --ring 3,2
        mode_kw = dict(mode_kw, ring_stages_cur=int(args.ring.split(",")[0]), ring_stages_prev=int(args.ring.split(",")[1]))
    if args.flags:                      # diagnostic: extra GFMC_FLAG_* bits for the main arm (e.g. 16 = GFMC_FLAG_NO_PDL for a same-box A/B)
        mode_kw = dict(mode_kw, flags=mode_kw.get("flags", 0) | args.flags)
    ctx = g.gfmc_create(L=L, M=M, t=cfg.t, JH=cfg.JH, T=cfg.T, mu=cfg.mu, n_energy=K, device=dev_index,
                        max_batch_sites=(-(-B // world) + 1) if shard else B, **mode_kw)
    g.gfmc_set_spins(ctx, S)

    # device-resident inputs for the `value` leg, pinned host buffers for the `e2e` leg
    d_batches = [torch.from_numpy(b).to(dev) for b in batches]
    d_prop = [torch.from_numpy(prop[0][b]).to(dev) for b in batches]
    d_uni = [torch.from_numpy(uni[0][b]).to(dev) for b in batches]
    h_sites = [torch.from_numpy(b).pin_memory() for b in batches]
    h_prop = [torch.from_numpy(np.ascontiguousarray(prop[0][b])).pin_memory() for b in batches]
    h_uni = [torch.from_numpy(np.ascontiguousarray(uni[0][b])).pin_memory() for b in batches]

    def step_device(i):
        j = i % len(batches)
        if shard:       # decide this rank's share, one all-gather of (accepted, dS) over NCCL, every rank applies all flips; device-resident throughout
            sharded.sharded_update_batch(ctx, d_batches[j], d_prop[j], d_uni[j], rank, world)
            ms_n = ctx.last_decide_loop_ms         # read inside, before gfmc_apply_flips resets the step-loop timing
        else:
            g.gfmc_update_batch(ctx, d_batches[j], d_prop[j], d_uni[j])
            ms_n = g.gfmc_last_step_loop_ms(ctx)   # CUDA events on the library's stream around the fused-step loop
        g.gfmc_magnetization(ctx)
        return ms_n

    def step_host(i):
        j = i % len(batches)
        if shard:
            dS, acc = sharded.sharded_update_batch(ctx, batches[j], prop[0][batches[j]], uni[0][batches[j]], rank, world,
                                                   device=dev if args.dist_backend == "nccl" else None)
        else:
            dS, acc = g.gfmc_update_batch(ctx, h_sites[j].numpy(), h_prop[j].numpy(), h_uni[j].numpy())
        return g.gfmc_magnetization(ctx), dS, acc

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    nvec = B if args.mode in ("ph", "ph2") else 2 * B       # start vectors propagated per batch
    happs_per_step = nvec * (M // 2)
    for i in range(args.warmup):
        step_device(i)
    sampler = ClockSampler(dev_index)
    sampler.start()
    c0 = g.gfmc_launch_counts(ctx)
    loop_ms, loop_steps = 0.0, 0
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(args.steps):
        ms, n = step_device(args.warmup + i)
        loop_ms += ms; loop_steps += n
    e1.record()
    barrier()
    elapsed = e0.elapsed_time(e1) * 1e-3
    c1 = g.gfmc_launch_counts(ctx)
    clocks = sampler.stop()
    # replicas: every rank did a whole batch per step (units add up); sharded: all ranks together did ONE batch per step
    my_units = float(happs_per_step * args.steps) / (world if shard else 1)
    t_max, units = aggregate_over_ranks(elapsed, my_units, world)
    n_chains = 1 if shard else world

    # e2e: same metric through the C ABI with HOST buffers (H2D of sites/proposals/uniforms and D2H of dS/accept/magnetization inside)
    if args.no_e2e:
        e2e_elapsed = float("nan")
    else:
        step_host(0)
        barrier()
        t0 = time.perf_counter()
        for i in range(args.steps):
            step_host(args.warmup + i)
        barrier()
        e2e_elapsed = time.perf_counter() - t0
    e2e_t, e2e_units = aggregate_over_ranks(e2e_elapsed, my_units, world)
    h2d = B * (4 + 24 + 8)
    d2h = B * (8 + 1) + 8

    if rank == 0:
        peak, peak_src = measured_peak()
        D = 2 * L ** 3
        dim = L ** 3 if args.mode == "dex" else D         # Eq. (2)-(3): one orbital per site
        alg_bytes = 48.0 * dim * nvec / (world if shard else 1)   # read r_{m-1}, read r_{m-2}, write r_m: 48 B per complex element (rank 0's launches)
        avg_launch_s = loop_ms * 1e-3 / max(loop_steps, 1)
        achieved = alg_bytes / avg_launch_s / 1e9 if avg_launch_s > 0.0 else float("nan")      # no timed step loop (e.g. an empty share): no figure
        line = {
            "metric": metric_name(cfg) + ("" if args.mode == "hund2" else f" [mode {args.mode}: not the headline]"), "value": units / t_max, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_max / args.steps * 1e3, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {cfg.index}: L={L} (D={D}) t={cfg.t} J_H={cfg.JH} T={cfg.T} mu={cfg.mu} M={M} K={K}, "
                                   f"{B}-site checkerboard batch ({nvec} start vectors) per step, uniform random spins seed {cfg.seed}",
                       "step": "gfmc_update_batch (a2-a7) + gfmc_magnetization (a8)",
                       "l2": f"inputs larger than L2: {2 * 16 * dim * nvec / 2**30:.1f} GiB of work vectors streamed every fused step",
                       "replicas": n_chains,
                       "parallelism": (f"one chain, every batch sharded over {world} GPUs, one all-gather of (accepted, dS) per batch" if shard
                                       else f"{world} independent chain(s), no data-path collective")},
            "site_updates_per_s": B * args.steps * n_chains / t_max,
            "clocks": clocks,
            "e2e": {"value": e2e_units / e2e_t, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "site_updates_per_s": B * args.steps * n_chains / e2e_t},
            "gpu_launches": (c1[0] - c0[0]) + (c1[1] - c0[1]),
            "roofline": {"bound": "hbm", "kernel": "cheb_step_kernel<false>", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "peak_source": peak_src, "traffic": ncu_traffic() if (args.mode == "hund2" and L == 32) else None,
                         "traffic_source": "committed ncu --set full capture of this kernel at config 4 (profiles/step_kernel_traffic.md); "
                                           "not measured in this run",
                         "algorithmic_bytes_per_launch": alg_bytes, "avg_launch_ms": avg_launch_s * 1e3,
                         "launches_timed": loop_steps, "step_loop_share_of_step": loop_ms * 1e-3 / elapsed},
        }
        if not args.no_copy_ref and world == 1 and L > 12:
            try:
                cp = sustained_copy_gbs(dev)
                line["roofline"]["copy_sustained_gbs_this_run"] = cp
                line["roofline"]["frac_of_sustained_copy"] = achieved / cp
            except RuntimeError as e:                           # not enough free memory beside the work vectors
                line["roofline"]["copy_sustained_gbs_this_run"] = None
                line["roofline"]["copy_sustained_note"] = str(e)[:120]
        if L <= 12:
            # small lattices run cheb_resident_kernel: the vectors never leave shared memory, so the bound is the
            # shared-memory pipe: 36 x 16 B accesses per site and fused step against 128 B/clk per SM at the clock measured under load
            nsm = torch.cuda.get_device_properties(dev_index).multi_processor_count
            smem_bytes = 36.0 * 16.0 * L ** 3 * B * (M // 2)                      # per batch (= per launch)
            sm_hz = (clocks.get("sm_mhz") or 1965.0) * 1e6
            smem_peak = nsm * 128.0 * sm_hz / 1e9
            per_launch_ms = loop_ms / max(args.steps, 1)                          # one launch per timed step (batch)
            ach = smem_bytes / (per_launch_ms * 1e-3) / 1e9
            line["config"]["l2"] = "vectors resident in shared memory for the whole recursion; no DRAM/L2 traffic for them"
            line["roofline"] = {"bound": "smem", "kernel": "cheb_resident_kernel", "achieved": ach, "peak": smem_peak, "unit": "GB/s",
                                "frac": ach / smem_peak, "peak_source": "128 B/clk/SM x SMs x SM clock sampled under load (DESIGN.md 5.5)",
                                "traffic": None, "algorithmic_bytes_per_launch": smem_bytes, "avg_launch_ms": per_launch_ms,
                                "launches_timed": args.steps, "step_loop_share_of_step": loop_ms * 1e-3 / elapsed}
        if not args.no_modes and world == 1 and args.mode == "hund2":
            g.gfmc_destroy(ctx)
            # same workload, same step, other modes of the fused kernel; not part of `value`
            ph = quick_mode_rate(cfg, B, dev_index, args.mode_steps, 2, ph_symmetry=1) if L % 2 == 0 else None
            if ph:
                # bytes the two-vector definition would have streamed per site update / time actually spent
                ph["effective_gbs_vs_two_vector_definition"] = 2.0 * ph["achieved_gbs"]
                ph["note"] = "Eq. (1), one start vector per site via A H A^-1 = -H (even L); same moments/decisions as the headline arm"
            dex = quick_mode_rate(cfg, B, dev_index, args.mode_steps, 2, model=g.GFMC_MODEL_DEX_INF)
            dex["note"] = ("Eq. (2)-(3) J_H->inf Hamiltonian (the paper's own runs), dimension N, start vectors |o>,|v> of Eq. (21); "
                           "same lattice, M, K, batch")
            line["modes"] = {"ph_symmetry": ph, "dex_inf": dex}
            if L == 32 and M % 4 == 0:
                ph2 = quick_mode_rate(cfg, B, dev_index, args.mode_steps, 2, ph_symmetry=1, flags=g.GFMC_FLAG_TWO_STEP)
                ph2["effective_gbs_vs_two_vector_definition"] = 2.0 * ph2["achieved_gbs"]
                ph2["note"] = ("ph_symmetry with TWO Chebyshev steps per pass over the vectors (temporal blocking, cheb_step2.cuh): 64 B of HBM traffic per "
                               "element and two steps instead of 96 B; achieved_gbs / frac count the ALGORITHMIC 48 B per element and step, so they "
                               "may exceed the HBM peak; avg_launch_ms is per fused STEP (half a launch)")
                line["modes"]["ph_two_step"] = ph2
            line["modes"]["exact_batch"] = exact_batch_rate(cfg, 32, dev_index, 3, 1)
            if cfg.index == 4 and not args.batch:
                # the two smaller single-GPU configurations, so that the driver's own run times them too (not part of `value`)
                line["configs"] = {"config3": config_leg(3, dev_index, 20, 3), "config2": config_leg(2, dev_index, 500, 20)}
        if not args.no_cpu and world == 1:
            cores = os.cpu_count() or 1
            v, desc = oracle_rate(cfg, 15.0, cores)
            v1, desc1 = oracle_rate(cfg, 6.0, 1)             # the same oracle on ONE core, beside the all-core figure
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                    "implied_site_updates_per_s": v / (2 * (M - 1)),
                                    "one_core": {"value": v1, "unit": UNIT, "cores": 1, "sample": desc1}}
        print(json.dumps(line), flush=True)
    if ctx.handle:
        g.gfmc_destroy(ctx)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def spawn_ranks(n: int) -> int:
    """Re-run this command line under torch.distributed.run with n ranks on this node (127.0.0.1 rendezvous on a free port)."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(Path(__file__).resolve()), *sys.argv[1:]]
    return subprocess.run(cmd, env=dict(os.environ, MASTER_ADDR="127.0.0.1")).returncode


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index (1-5); 4 = the headline L=32 workload")
    ap.add_argument("--batch", type=int, default=0, help="override the batch size (sites)")
    ap.add_argument("--impl", default="gfmc", choices=["gfmc", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-modes", action="store_true", help="skip the extra ph_symmetry / dex_inf measurements")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: shard ONE chain's batches over the ranks (SURVEY.md 8(e), strong scaling) instead of N independent replicas")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="N > 1: nccl = one rank per GPU; gloo = host-staged exchange, ranks wrap around the GPUs present (tests on a one-GPU box)")
    ap.add_argument("--no-copy-ref", action="store_true", help="skip the 1.5 s sustained-copy measurement reported beside the roofline fraction")
    ap.add_argument("--ring", default="", help="diagnostic: ring depths C,P of the streaming kernel (default: automatic)")
    ap.add_argument("--flags", type=int, default=0, help="diagnostic: GFMC_FLAG_* bits OR-ed into the main arm's context flags (16 = no programmatic dependent launch)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs only; the contract line needs it)")
    ap.add_argument("--mode", default="hund2", choices=["hund2", "ph", "ph2", "dex"],
                    help="mode of the fused kernel the main arm times; hund2 = the headline (two start vectors per site, Eq. (1))")
    ap.add_argument("--mode-steps", type=int, default=5, help="timed steps of each extra mode (after 2 warm-up steps)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N ranks ourselves, exactly as the driver's torchrun line does
        sys.exit(spawn_ranks(args.gpus))
    from paper_1303_6016_b200 import workload as wl
    cfg = wl.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_gfmc(args, cfg)


if __name__ == "__main__":
    main()
