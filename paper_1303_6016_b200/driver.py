"""Host-side driver of SURVEY.md §8(f3): magnetization versus temperature with Algorithm 1 (the paper's
validation runs, Fig. 4).  Orchestration only -- every number comes from libgfmc.so (gfmc_run draws the trial
moves on the device, gfmc_set_temperature changes beta); one context anneals through the temperature list.
"""
from __future__ import annotations

import os

import numpy as np

from . import binding as g
from . import workload as wl


def magnetization_curve(L: int, M: int, temperatures, n_warmup: int, n_measure: int, batch_sites: int, seed: int = 1,
                        t: float = 1.0, JH: float = 8.0, mu: float = 0.0, n_energy: int = 0, model: int = g.GFMC_MODEL_HUND,
                        ph_symmetry: int = 0, spins=None, device: int = 0):
    """For each T in `temperatures` (in the given order, each starting from the previous configuration): n_warmup sweeps, then
    n_measure sweeps whose |sum_i S_i|/N is averaged (Alg. 1 lines 14-17).  Sweep indices run on across temperatures, so the
    whole scan is one reproducible chain of `seed`.  Returns dict(T, m_mean, m_err, acceptance, series, spins)."""
    temperatures = [float(T) for T in temperatures]
    S0 = wl.make_spins(L, seed) if spins is None else np.asarray(spins, dtype=np.float64)
    ctx = g.gfmc_create(L=L, M=M, t=t, JH=JH, T=temperatures[0], mu=mu, n_energy=n_energy, max_batch_sites=batch_sites,
                        device=device, model=model, ph_symmetry=ph_symmetry)
    try:
        g.gfmc_set_spins(ctx, S0)
        sweep, out = 0, dict(T=[], m_mean=[], m_err=[], acceptance=[], series=[])
        for T in temperatures:
            g.gfmc_set_temperature(ctx, T)
            if n_warmup:
                g.gfmc_run(ctx, seed, sweep, n_warmup, batch_sites)
                sweep += n_warmup
            mag, nacc = g.gfmc_run(ctx, seed, sweep, n_measure, batch_sites)
            sweep += n_measure
            st = g.gfmc_run_summary(ctx)          # Alg. 1 lines 16-17: averaged by the library, on the device
            out["T"].append(T); out["m_mean"].append(st["mean"]); out["m_err"].append(st["stderr"])
            out["acceptance"].append(st["acceptance"]); out["series"].append(mag)
        out["spins"] = g.gfmc_get_spins(ctx)
        return out
    finally:
        g.gfmc_destroy(ctx)


def magnetization_curve_parallel(L: int, M: int, temperatures, n_warmup: int, n_measure: int, batch_sites: int, seed: int = 1,
                                 t: float = 1.0, JH: float = 8.0, mu: float = 0.0, n_energy: int = 0, model: int = g.GFMC_MODEL_HUND,
                                 ph_symmetry: int = 0, spins=None, device: int = 0, max_workers: int = 0):
    """The paper's own parallel level (independent Monte Carlo chains, no communication) on ONE GPU: every
    temperature is an independent chain (seed + index, same start configuration) with its own context and CUDA stream, driven from
    its own host thread, so the chains' kernels overlap on the GPU.  Meant for the sequential regime (small batch_sites on small
    lattices), where one chain keeps one SM busy and leaves the other 147 idle.  Unlike magnetization_curve the chains are not
    annealed into each other: every temperature warms up from `spins` (default: the seeded random configuration).
    Returns the same dict (spins: list, one final configuration per temperature)."""
    import concurrent.futures as cf
    # Concurrent chains need one hardware work queue per stream to overlap; the CUDA default is 8.  The variable is read when the
    # process initialises CUDA, so it only helps if this function runs before the first CUDA call of the process (torch initialises
    # CUDA lazily); a value the caller has set is left alone.  Set here, not at import: importing the package changes nothing.
    os.environ.setdefault("CUDA_DEVICE_MAX_CONNECTIONS", "32")
    import torch
    temperatures = [float(T) for T in temperatures]
    S0 = wl.make_spins(L, seed) if spins is None else np.asarray(spins, dtype=np.float64)

    def chain(idx_T):
        idx, T = idx_T
        torch.cuda.set_device(device)
        # stream 0 = "no stream given": the library creates one stream per context (torch's stream pool would hand the same
        # stream to every 32nd chain, which serialises them and cannot be captured by two contexts at once)
        ctx = g.gfmc_create(L=L, M=M, t=t, JH=JH, T=T, mu=mu, n_energy=n_energy, max_batch_sites=batch_sites, device=device,
                            stream=0, model=model, ph_symmetry=ph_symmetry)
        try:
            g.gfmc_set_spins(ctx, S0)
            if n_warmup:
                g.gfmc_run(ctx, seed + idx, 0, n_warmup, batch_sites)
            mag, nacc = g.gfmc_run(ctx, seed + idx, n_warmup, n_measure, batch_sites)
            return T, mag, g.gfmc_run_summary(ctx), g.gfmc_get_spins(ctx)
        finally:
            g.gfmc_destroy(ctx)

    workers = max_workers or len(temperatures)
    with cf.ThreadPoolExecutor(max_workers=workers) as pool:
        results = list(pool.map(chain, enumerate(temperatures)))
    out = dict(T=[], m_mean=[], m_err=[], acceptance=[], series=[], spins=[])
    for T, mag, st, S in results:
        out["T"].append(T); out["m_mean"].append(st["mean"]); out["m_err"].append(st["stderr"])
        out["acceptance"].append(st["acceptance"]); out["series"].append(mag); out["spins"].append(S)
    return out


def main(argv=None):
    """python -m paper_1303_6016_b200.driver --L 6 --M 256 --T 0.3 0.2 0.15 0.12 0.1 0.08 0.05 --warmup 150 --measure 250 --batch 1 --model dex"""
    import argparse
    import json
    import time
    ap = argparse.ArgumentParser(description="magnetization versus temperature with Algorithm 1 (arXiv:1303.6016) on one B200")
    ap.add_argument("--L", type=int, default=6)
    ap.add_argument("--M", type=int, default=256, help="Chebyshev truncation number (the paper's validation uses 256)")
    ap.add_argument("--T", type=float, nargs="+", default=[0.30, 0.20, 0.15, 0.12, 0.10, 0.08, 0.05])
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--measure", type=int, default=50)
    ap.add_argument("--batch", type=int, default=1, help="sites per frozen batch; 1 = the paper's sequential algorithm")
    ap.add_argument("--model", choices=["dex", "hund"], default="dex", help="dex: J_H->inf, Eq. (2)-(3); hund: Eq. (1)")
    ap.add_argument("--JH", type=float, default=8.0)
    ap.add_argument("--mu", type=float, default=0.0)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--parallel", action="store_true", help="one independent chain per temperature, all concurrently on the GPU")
    ap.add_argument("--json", default="", help="also write the result to this file")
    a = ap.parse_args(argv)
    t0 = time.time()
    fn = magnetization_curve_parallel if a.parallel else magnetization_curve
    r = fn(a.L, a.M, a.T, a.warmup, a.measure, a.batch, seed=a.seed, JH=a.JH, mu=a.mu,
           model=g.GFMC_MODEL_DEX_INF if a.model == "dex" else g.GFMC_MODEL_HUND)
    print(f"# L={a.L} M={a.M} model={a.model} batch={a.batch} warmup={a.warmup} measure={a.measure} seed={a.seed}: {time.time() - t0:.1f} s")
    print("#     T        m     stderr  acceptance")
    for T, m, e, acc in zip(r["T"], r["m_mean"], r["m_err"], r["acceptance"]):
        print(f"{T:8.4f} {m:8.4f} {e:8.4f} {acc:8.4f}")
    if a.json:
        with open(a.json, "w") as f:
            json.dump({k: (v if k != "series" else [s.tolist() for s in v]) for k, v in r.items() if k != "spins"}, f)


if __name__ == "__main__":
    main()
