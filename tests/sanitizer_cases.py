"""Small invocations for `compute-sanitizer --tool memcheck|racecheck python -m tests.sanitizer_cases` (profiles/r2_sanitizer.md; the tool
is closed on this pool, so tests/test_gpu_determinism.py runs them as a plain GPU test and stands in for racecheck with bitwise
repeatability across ring depths).  Test infrastructure, not part of the product's entry module."""
import sys
from pathlib import Path

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))


def sanitizer_cases() -> None:
    """Small invocations that exercise every synchronisation protocol of the kernels, meant to run under
    `compute-sanitizer --tool memcheck|racecheck` (profiles/r2_sanitizer.md): the streaming kernel with the balanced work list
    (L = 16: mbarrier stage release + CAS-claimed refill + per-warp R_prev / bond rings + in-place overwrite of r_{m-2}), the
    run-time-L streaming kernel (L = 20: CTA-wide R_prev ring) and the shared-memory-resident kernel (L = 8), in all three modes,
    followed by one frozen-batch update each."""
    import numpy as np
    import paper_1303_6016_b200 as g
    from paper_1303_6016_b200 import workload as wl
    for L, M, n in ((16, 8, 512), (20, 6, 150), (8, 8, 64)):
        S = wl.make_spins(L, seed=L)
        rng = np.random.default_rng(L)
        sites = np.sort(rng.choice(L ** 3, size=n, replace=False)).astype(np.int32)
        prop = wl.make_spins(L, seed=L + 1)[sites]
        uni = 1.0 - rng.random(n)
        for name, kw in (("hund", {}), ("ph", dict(ph_symmetry=1)), ("dex", dict(model=g.GFMC_MODEL_DEX_INF))):
            ctx = g.gfmc_create(L=L, M=M, t=1.0, JH=4.0, T=0.05, max_batch_sites=n, **kw)
            g.gfmc_set_spins(ctx, S)
            mu = g.gfmc_moments_ov(ctx, sites, prop) if name == "dex" else g.gfmc_moments(ctx, sites)
            dS, acc = g.gfmc_update_batch(ctx, sites, prop, uni)
            print(f"sanitizer case L={L} {name}: |mu|max={np.abs(mu).max():.3f} accepted={int(acc.sum())}/{n} "
                  f"launches={g.gfmc_launch_counts(ctx)}", flush=True)
            g.gfmc_destroy(ctx)


if __name__ == "__main__":
    sanitizer_cases()
