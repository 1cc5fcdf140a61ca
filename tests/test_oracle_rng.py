"""Pins of oracle/rng.py (the counter-based generator of the Algorithm-1 driver, reading f3-1)."""
from pathlib import Path

import numpy as np

from oracle import rng

GOLDEN = Path(__file__).parent / "golden" / "philox4x32_10_kat.txt"


def test_philox_known_answers():
    rows = [l.split() for l in GOLDEN.read_text().splitlines() if l and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        out = rng.philox4x32_10(w[0:4], w[4:6])
        assert [int(o[0]) for o in out] == w[6:10]


def test_philox_is_elementwise():
    """vectorised call == one call per counter (the site index is the only word that varies inside a sweep)"""
    sites = np.arange(50)
    v = rng.philox4x32_10((sites, np.full(50, 7), np.ones(50), np.zeros(50)), (123, 456))
    for i in (0, 1, 17, 49):
        s = rng.philox4x32_10((i, 7, 1, 0), (123, 456))
        assert [int(x[0]) for x in s] == [int(x[i]) for x in v]


def test_uniform_conversion_range_and_resolution():
    assert rng._u01(np.uint64(0), np.uint64(0))[()] == 0.0
    top = rng._u01(np.uint64(0xFFFFFFFF), np.uint64(0xFFFFFFFF))
    assert top < 1.0 and top == 1.0 - 2.0 ** -53
    assert rng._u01(np.uint64(0x80000000), np.uint64(0)) == 0.5


def test_proposals_are_unit_vectors_uniform_on_the_sphere():
    N = 200_000
    S, u = rng.proposals(seed=2026, sweep=3, N=N)
    assert np.abs(np.linalg.norm(S, axis=1) - 1.0).max() < 4e-16
    assert u.min() > 0.0 and u.max() <= 1.0
    # first and second moments of a uniform distribution on the sphere: <S> = 0, <S_a S_b> = delta_ab / 3; <u> = 1/2, var = 1/12
    assert np.abs(S.mean(axis=0)).max() < 5 / np.sqrt(3 * N)
    C = S.T @ S / N
    assert np.abs(C - np.eye(3) / 3).max() < 5 / np.sqrt(N)
    assert abs(u.mean() - 0.5) < 5 / np.sqrt(12 * N) and abs(u.var() - 1 / 12) < 5e-3
    # different sweeps, seeds and streams are different numbers
    S2, u2 = rng.proposals(seed=2026, sweep=4, N=N)
    S3, u3 = rng.proposals(seed=2027, sweep=3, N=N)
    assert not np.array_equal(S, S2) and not np.array_equal(S, S3) and not np.array_equal(u, u2) and not np.array_equal(u, u3)
    assert abs(np.corrcoef(u, u2)[0, 1]) < 5 / np.sqrt(N) and abs(np.corrcoef(S[:, 2], u)[0, 1]) < 5 / np.sqrt(N)


def test_sweep_index_above_32_bits_uses_the_fourth_counter_word():
    a = rng.uniforms(1, (1 << 32) + 5, 8)
    b = rng.uniforms(1, 5, 8)
    assert not np.array_equal(a[0], b[0])
    w = rng.philox4x32_10((3, 5, 0, 1), (1, 0))
    assert a[0][3] == rng._u01(w[0], w[1])[0]


def test_run_chain_feeds_the_oracle_sweep():
    """run_chain == calling oracle.sweep once with the stacked generator outputs (L=4, 2 sweeps)."""
    from oracle import oracle
    from paper_1303_6016_b200 import workload as wl
    L, M, K, B = 4, 16, 32, 4
    S = wl.make_spins(L, seed=11)
    fn = lambda S_, p, u: oracle.sweep(L, 1.0, 4.0, 0.05, 0.0, M, K, 0, 4.0, S_, 1, B, p, u, nthreads=2)
    r = rng.run_chain(fn, S, seed=5, first_sweep=10, n_sweeps=2)
    P = np.stack([rng.proposals(5, 10, L ** 3)[0], rng.proposals(5, 11, L ** 3)[0]])
    U = np.stack([rng.proposals(5, 10, L ** 3)[1], rng.proposals(5, 11, L ** 3)[1]])
    ref = oracle.sweep(L, 1.0, 4.0, 0.05, 0.0, M, K, 0, 4.0, S, 2, B, P, U, nthreads=2)
    assert np.array_equal(r["spins"], ref["spins"]) and np.array_equal(r["accept"], ref["accept"])
    assert np.array_equal(r["magnetization"], ref["magnetization"]) and np.array_equal(r["dS"], ref["dS"])
