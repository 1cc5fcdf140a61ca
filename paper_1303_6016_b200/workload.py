"""Seeded synthetic workload generator (serves BOTH the CUDA path and the oracle).

This module holds none of the method's arithmetic: it only draws classical-spin
fields, trial spins and Metropolis uniforms from a seeded stream, in the shapes of
the paper's runs (simple-cubic lattices, |S_i| = 1; "change the
spin randomly", Algorithm 1 line 3; "rand()", line 10,
PAPER.md:292).  It stands in for the paper's Monte Carlo configurations, which
are not published.

Recipe: ``numpy.random.default_rng(seed)``, only ``.random()``
doubles, in this draw order:
  1. spins: two uniforms (u1, u2) per site, site order i = x + L*(y + L*z);
  2. for every sweep, for every site: (u1, u2) for the proposal, u3 for the
     acceptance test; the library receives ``u = 1 - u3`` in (0, 1] so that
     ``ln u`` is finite.
Uniform on the sphere: z = 2*u1 - 1, phi = 2*pi*u2.
Cone of half-angle alpha about +z (uniform on the cap): z = 1 - u1*(1 - cos alpha).
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np


@dataclass(frozen=True)
class Config:
    """One of BASELINE.json's ``configs`` (index 1..5), see SURVEY.md §8(d)."""
    index: int
    L: int
    t: float
    JH: float
    T: float
    mu: float
    spins: str          # "sphere" | "cone"
    cone: float         # half-angle in rad (cone only)
    seed: int
    M: int
    K: int              # energy points, 2*M (SURVEY.md §8(c) reading 10)
    batch_sites: int    # B for gfmc_sweep
    sweeps: int

    @property
    def N(self) -> int:
        return self.L ** 3

    @property
    def D(self) -> int:
        return 2 * self.L ** 3


CONFIGS = {
    1: Config(1, 4, 1.0, 4.0, 0.05, 0.0, "sphere", 0.0, 1, 64, 128, 1, 1),
    2: Config(2, 8, 1.0, 4.0, 0.05, 0.0, "sphere", 0.0, 2, 256, 512, 256, 10),
    3: Config(3, 16, 1.0, 8.0, 0.02, 0.0, "cone", 0.6, 3, 512, 1024, 512, 10),
    4: Config(4, 32, 1.0, 8.0, 0.02, 0.0, "sphere", 0.0, 4, 1024, 2048, 2048, 5),
    5: Config(5, 64, 1.0, 8.0, 0.01, 0.0, "cone", 0.3, 5, 2048, 4096, 4096, 2),
}


def _unit_vectors(u1: np.ndarray, u2: np.ndarray, kind: str, cone: float) -> np.ndarray:
    if kind == "sphere":
        z = 2.0 * u1 - 1.0
    elif kind == "cone":
        z = 1.0 - u1 * (1.0 - np.cos(cone))
    else:
        raise ValueError(f"unknown spin distribution {kind!r}")
    phi = 2.0 * np.pi * u2
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    out = np.empty(u1.shape + (3,), dtype=np.float64)
    out[..., 0] = s * np.cos(phi)
    out[..., 1] = s * np.sin(phi)
    out[..., 2] = z
    # exact unit length to rounding (the library validates | |S|-1 | <= 1e-12)
    out /= np.linalg.norm(out, axis=-1, keepdims=True)
    return out


def make_spins(L: int, seed: int, kind: str = "sphere", cone: float = 0.0,
               rng: np.random.Generator | None = None) -> np.ndarray:
    """Spin field [N,3] fp64; consumes 2 uniforms per site from ``rng``."""
    rng = np.random.default_rng(seed) if rng is None else rng
    u = rng.random((L ** 3, 2))
    return np.ascontiguousarray(_unit_vectors(u[:, 0], u[:, 1], kind, cone))


def make_workload(cfg: Config, n_sweeps: int | None = None):
    """Returns (spins [N,3], proposals [S,N,3], uniforms [S,N] in (0,1])."""
    S = cfg.sweeps if n_sweeps is None else n_sweeps
    rng = np.random.default_rng(cfg.seed)
    spins = make_spins(cfg.L, cfg.seed, cfg.spins, cfg.cone, rng=rng)
    proposals = np.empty((S, cfg.N, 3), dtype=np.float64)
    uniforms = np.empty((S, cfg.N), dtype=np.float64)
    for s in range(S):
        u = rng.random((cfg.N, 3))
        # proposals are uniform on the sphere, independent of the current spin
        proposals[s] = _unit_vectors(u[:, 0], u[:, 1], "sphere", 0.0)
        uniforms[s] = 1.0 - u[:, 2]
    return spins, proposals, uniforms


def ferromagnet(L: int, nhat=(0.0, 0.0, 1.0)) -> np.ndarray:
    n = np.asarray(nhat, dtype=np.float64)
    n = n / np.linalg.norm(n)
    return np.ascontiguousarray(np.tile(n, (L ** 3, 1)))


def neel(L: int) -> np.ndarray:
    """S_i = (-1)^(x+y+z) z-hat (L even for a consistent periodic pattern)."""
    idx = np.arange(L ** 3)
    x, y, z = idx % L, (idx // L) % L, idx // (L * L)
    sgn = 1.0 - 2.0 * ((x + y + z) % 2)
    S = np.zeros((L ** 3, 3), dtype=np.float64)
    S[:, 2] = sgn
    return S


def colour_sites(L: int, colour: int) -> np.ndarray:
    """Sites of checkerboard colour (x+y+z) mod 2, increasing index (int32)."""
    idx = np.arange(L ** 3)
    x, y, z = idx % L, (idx // L) % L, idx // (L * L)
    return idx[((x + y + z) % 2) == colour].astype(np.int32)


def sha256(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
