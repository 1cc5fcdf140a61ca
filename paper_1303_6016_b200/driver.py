"""Host-side driver of SURVEY.md §8(f3): magnetization versus temperature with Algorithm 1 (the paper's
validation runs, Fig. 4).  Orchestration only -- every number comes from libgfmc.so (gfmc_run draws the trial
moves on the device, gfmc_set_temperature changes beta); one context anneals through the temperature list.
"""
from __future__ import annotations

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
            out["T"].append(T); out["m_mean"].append(float(mag.mean()))
            out["m_err"].append(float(mag.std(ddof=1) / np.sqrt(len(mag))) if len(mag) > 1 else float("nan"))
            out["acceptance"].append(float(nacc.sum()) / (len(mag) * ctx.N)); out["series"].append(mag)
        out["spins"] = g.gfmc_get_spins(ctx)
        return out
    finally:
        g.gfmc_destroy(ctx)
