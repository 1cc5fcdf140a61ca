"""Host-side checks of the seeded workload generator (no oracle arithmetic, no CUDA)."""
from pathlib import Path

import numpy as np

from paper_1303_6016_b200 import workload as wl

GOLD = Path(__file__).resolve().parent / "golden"


def test_unit_length_and_ranges():
    for i in (1, 2, 3):
        cfg = wl.CONFIGS[i]
        S, prop, uni = wl.make_workload(cfg, n_sweeps=2)
        assert S.shape == (cfg.N, 3) and prop.shape == (2, cfg.N, 3) and uni.shape == (2, cfg.N)
        assert np.abs(np.linalg.norm(S, axis=-1) - 1).max() < 1e-15
        assert np.abs(np.linalg.norm(prop, axis=-1) - 1).max() < 1e-15
        assert uni.min() > 0.0 and uni.max() <= 1.0


def test_cone_distribution():
    cfg = wl.CONFIGS[3]
    S, _, _ = wl.make_workload(cfg, n_sweeps=1)
    assert S[:, 2].min() >= np.cos(0.6) - 1e-15
    # uniform on the cap: z uniform in [cos(alpha), 1]
    assert abs(S[:, 2].mean() - (1 + np.cos(0.6)) / 2) < 0.01


def test_sphere_distribution_moments():
    S = wl.make_spins(16, seed=11)
    assert np.abs(S.mean(0)).max() < 0.03 and np.abs((S ** 2).mean(0) - 1 / 3).max() < 0.02


def test_seeded_and_stable():
    a = wl.make_workload(wl.CONFIGS[2], n_sweeps=1)
    b = wl.make_workload(wl.CONFIGS[2], n_sweeps=1)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    # more sweeps extend the stream without changing the prefix
    c = wl.make_workload(wl.CONFIGS[2], n_sweeps=2)
    assert np.array_equal(a[1][0], c[1][0]) and np.array_equal(a[2][0], c[2][0])


def test_golden_hashes():
    want = {}
    for line in (GOLD / "workload_sha256.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        cfg, name, h = line.split()
        want[(cfg, name)] = h
    for i in (1, 2, 3):
        S, prop, uni = wl.make_workload(wl.CONFIGS[i], n_sweeps=1)
        assert want[(f"cfg{i}", "spins")] == wl.sha256(S)
        assert want[(f"cfg{i}", "proposals")] == wl.sha256(prop)
        assert want[(f"cfg{i}", "uniforms")] == wl.sha256(uni)


def test_oracle_golden_moments(oracle):
    cfg = wl.CONFIGS[1]
    S, _, _ = wl.make_workload(cfg, n_sweeps=1)
    mu = oracle.moments(cfg.L, cfg.t, cfg.JH, S, site=21, M=16)
    for line in (GOLD / "oracle_cfg1_moments.txt").read_text().splitlines():
        if line.startswith("#"):
            continue
        n, al, be, re, im = line.split()
        assert abs(mu[int(n), int(al), int(be)] - complex(float(re), float(im))) < 1e-14


def test_colour_sites_and_states():
    L = 4
    c0, c1 = wl.colour_sites(L, 0), wl.colour_sites(L, 1)
    assert len(c0) == len(c1) == 32 and set(c0) | set(c1) == set(range(64))
    assert c0.dtype == np.int32 and np.all(np.diff(c0) > 0)
    assert np.array_equal(wl.neel(L)[c0, 2], np.ones(32)) and np.array_equal(wl.neel(L)[c1, 2], -np.ones(32))
    assert np.allclose(np.linalg.norm(wl.ferromagnet(3, (1, 2, 2)), axis=1), 1.0)
