"""Pins for oracle/gfmc_oracle_exact.c (exactness inside a batch).  No CUDA here.

The oracle's claim is the Dyson/Woodbury identity G_U,BB = G_BB - G_BU Delta_U (1 + G_UU Delta_U)^-1 G_UB inside
d = Det[1 + G Delta] (Eq. (11)).  It is pinned against what the mathematics fixes, not against itself:
eigenvalue products of dense matrices (Eq. (12)), dense eigen-moments, and the paper's own sequential
Algorithm 1 as the limit the batch must reproduce."""
import numpy as np
import pytest

from paper_1303_6016_b200 import workload as wl
from tests.dense import SIGMA, cheb_T, dense_H


def _a(t, JH):
    return 6 * abs(t) + np.sqrt(2.0) * abs(JH)


def _delta(JH, S_old, S_new):
    return JH * np.einsum("c,cab->ab", S_new - S_old, SIGMA)


def _embed(D, site, blk):
    out = np.zeros((D, D), dtype=np.complex128)
    out[2 * site:2 * site + 2, 2 * site:2 * site + 2] = blk
    return out


# ------------------------------------------------------------------ cross moments (pin 2)
@pytest.mark.parametrize("L", [3, 4])
def test_cross_moments_against_dense_eigendecomposition(oracle, L):
    t, JH, M = 1.0, 4.0, 40
    S = wl.make_spins(L, seed=20 + L)
    sites = np.array([0, 5, L ** 3 - 1, 7], dtype=np.int32)
    mu = oracle.cross_moments(L, t, JH, S, sites, M, nthreads=2)
    a = _a(t, JH)
    e, V = np.linalg.eigh(dense_H(L, t, JH, S))
    Tn = np.stack([cheb_T(n, e / a) for n in range(M)])                        # [M, D]
    for X, sx in enumerate(sites):
        for Y, sy in enumerate(sites):
            for al in range(2):
                for be in range(2):
                    ref = (Tn * (V[2 * sx + al, :] * V[2 * sy + be, :].conj())[None, :]).sum(axis=1)
                    assert np.abs(mu[X, Y, :, al, be] - ref).max() < 5e-14
    # Hermiticity of T_m(H~): mu(X,Y) = mu(Y,X)^dagger; diagonal blocks are the single-site moments
    assert np.abs(mu - mu.transpose(1, 0, 2, 4, 3).conj()).max() < 1e-14
    for X, sx in enumerate(sites):
        assert np.array_equal(mu[X, X], oracle.moments(L, t, JH, S, int(sx), M))
    # mu_0 = identity between equal sites, 0 otherwise
    for X in range(4):
        for Y in range(4):
            assert np.array_equal(mu[X, Y, 0], np.eye(2) if X == Y else np.zeros((2, 2)))


# ------------------------------------------------------------------ the Dyson step with the exact resolvent (pin 1)
@pytest.mark.parametrize("L,pattern", [(3, "all"), (4, "all"), (4, "mixed")])
def test_conditional_determinants_equal_eigenvalue_products(oracle, L, pattern):
    """Exact resolvent blocks in, conditional d_B|U(z) out: must equal det(H + Delta_U + Delta_B - z)/det(H + Delta_U - z)
    (Eq. (12)) for the accepted set U the oracle itself reports; the product over the batch is the joint ratio."""
    t, JH, T = 1.0, 4.0, 0.3
    S = wl.make_spins(L, seed=30 + L)
    N, D = L ** 3, 2 * L ** 3
    a = _a(t, JH)
    sites = np.array([0, 2, 9, 11, N - 1], dtype=np.int32) if L == 4 else np.array([0, 1, 13, 26], dtype=np.int32)   # L = 3: neighbours too
    n = len(sites)
    S_new = wl.make_spins(L, seed=31 + L)[sites]
    S_new[1] = S[sites[1]]                                                     # one trial that changes nothing
    K = 24
    phi = np.pi * (np.arange(K) + 0.5) / K
    z = a * np.cos(phi) + 0.37j * (1.0 + np.sin(3 * phi))                     # complex energies, away from the spectrum
    H = dense_H(L, t, JH, S)
    rows = np.concatenate([[2 * s, 2 * s + 1] for s in sites])
    Gt = np.empty((n, n, K, 2, 2), dtype=np.complex128)
    for k in range(K):
        G = np.linalg.inv(H - z[k] * np.eye(D))[np.ix_(rows, rows)]           # Eq. (10): G = 1/(H - z)
        Gt[:, :, k] = a * G.reshape(n, 2, n, 2).transpose(0, 2, 1, 3)         # G~ = a G
    uni = np.full(n, 1e-300) if pattern == "all" else np.array([1e-300, 1.0, 1.0, 1e-300, 1.0])[:n]
    dS, acc, d = oracle.exact_batch(Gt, S[sites], S_new, uni, JH, a, 0.0, T, 0.0, want_d=True)
    if pattern == "all":
        assert acc.all()
    Hc = H.copy()
    joint = np.ones(K, dtype=np.complex128)
    for B in range(n):
        Hn = Hc + _embed(D, sites[B], _delta(JH, S[sites[B]], S_new[B]))
        ref = np.array([np.prod((np.linalg.eigvalsh(Hn) - zk) / (np.linalg.eigvalsh(Hc) - zk)) for zk in z])
        assert np.abs(d[B] - ref).max() <= 1e-12 * np.abs(ref).max(), (B, np.abs(d[B] - ref).max())
        if acc[B]:
            Hc = Hn
            joint *= d[B]
    Hall = H + sum(_embed(D, sites[B], _delta(JH, S[sites[B]], S_new[B])) for B in range(n) if acc[B])
    ref_joint = np.array([np.prod((np.linalg.eigvalsh(Hall) - zk) / (np.linalg.eigvalsh(H) - zk)) for zk in z])
    assert np.abs(joint - ref_joint).max() <= 1e-11 * np.abs(ref_joint).max()
    assert np.all(d[1] == 1.0) and dS[1] == 0.0                                # S' = S: d = 1 exactly


# ------------------------------------------------------------------ frozen batch as the special case (pin 4)
def test_no_accepted_change_is_the_frozen_batch_bit_for_bit(oracle):
    L, t, JH, T, M, K = 4, 1.0, 4.0, 0.05, 48, 96
    S = wl.make_spins(L, seed=40)
    sites = wl.colour_sites(L, 0)[:6]
    prop = wl.make_spins(L, seed=41)[sites]
    frozen = np.array([oracle.site_dS(L, t, JH, T, 0.0, M, K, 0, 4.0, S, int(s), prop[j]) for j, s in enumerate(sites)])
    # (i) every trial rejected: u = 1 accepts only Delta S < 0, so use the frozen values to pick the rejected ones
    rej = frozen > 0
    assert rej.sum() >= 2
    dS, acc = oracle.exact_batch_dS(L, t, JH, T, 0.0, M, K, 0, 4.0, S, sites[rej], prop[rej], np.ones(int(rej.sum())))
    assert not acc.any() and np.array_equal(dS, frozen[rej])
    # (ii) accepted trials that change nothing (S' = S) in front of real ones
    sites2 = np.array([sites[0], sites[1], sites[2], sites[3]], dtype=np.int32)
    prop2 = np.stack([S[sites[0]], S[sites[1]], prop[2], prop[3]])
    dS2, acc2 = oracle.exact_batch_dS(L, t, JH, T, 0.0, M, K, 0, 4.0, S, sites2, prop2, np.array([0.5, 0.5, 1.0, 1.0]))
    assert acc2[0] and acc2[1] and dS2[0] == 0.0 and dS2[1] == 0.0
    assert dS2[2] == frozen[2]
    if not acc2[2]:
        assert dS2[3] == frozen[3]


# ------------------------------------------------------------------ the sequential algorithm as the limit (pin 3)
def _pair_errors(oracle, L, T, kernel, Ms):
    """Sites A, B of one batch, A accepted (a full reversal: the largest Delta).  Returns, per M, |Delta S_B(exact batch) -
    Delta S_B(sequential)| and |Delta S_B(frozen batch) - Delta S_B(sequential)|, sequential = a fresh recursion with A flipped."""
    t, JH = 1.0, 4.0
    S = wl.make_spins(L, seed=50)
    A, B = 0, 2                                                                 # same colour, second neighbours along x
    prop = wl.make_spins(L, seed=51)[[A, B]]
    prop[0] = -S[A]
    S_seq = S.copy(); S_seq[A] = prop[0]
    err_exact, err_frozen = [], []
    for M in Ms:
        K = 2 * M
        seq = oracle.site_dS(L, t, JH, T, 0.0, M, K, kernel, 4.0, S_seq, B, prop[1])
        frozen = oracle.site_dS(L, t, JH, T, 0.0, M, K, kernel, 4.0, S, B, prop[1])
        dS, acc = oracle.exact_batch_dS(L, t, JH, T, 0.0, M, K, kernel, 4.0, S, np.array([A, B], dtype=np.int32), prop,
                                        np.array([1e-300, 0.5]), nthreads=2)
        assert acc[0]
        err_exact.append(abs(dS[1] - seq)); err_frozen.append(abs(frozen - seq))
    return np.array(err_exact), np.array(err_frozen)


@pytest.mark.parametrize("L,T", [(4, 0.05), (4, 0.5), (6, 0.05)])
def test_two_site_batch_reproduces_the_sequential_chain_lorentz_kernel(oracle, L, T):
    """Sequential Algorithm 1 evaluates B with A's new spin in H (a fresh recursion); the exact batch gets there by the Dyson
    update of the batch-start G.  The Lorentz-damped series (the paper's kernel) is the resolvent at a complex
    energy E + i eps(E) up to the truncation, and the Dyson identity holds at every complex energy: the two agree up to a
    truncation error that shrinks like 1/M, while the frozen batch keeps its O(G_AB^2) error whatever M is."""
    err_exact, err_frozen = _pair_errors(oracle, L, T, 1, (64, 256, 1024))
    assert err_exact[0] > err_exact[1] > err_exact[2]
    assert err_exact[2] < 0.35 * err_exact[1] < 0.35 * 0.6 * err_exact[0]       # ~ 1/M (measured: factor 3-4 per factor 4 in M)
    assert err_exact[2] < 0.02 * err_frozen[2], (err_exact, err_frozen)
    assert err_frozen.min() > 1e-3 * (1.0 if T < 0.1 else 0.1)                  # the frozen-batch error is real and does not shrink


def test_two_site_batch_jackson_kernel_while_levels_are_not_resolved(oracle):
    """A Jackson-damped series is a convolution with a near-Gaussian, not a resolvent at a complex energy, so the Dyson identity
    holds only while the broadening (~ pi a / M) stays above the level spacing (~ 2a/D): at L = 6 (D = 432) and M <= 256 the
    exact batch is 10-100 x closer to the sequential chain than the frozen batch.  (At L = 4, M = 1024, where single levels
    are resolved, it is not -- DESIGN.md says so; production lattices have D >= 8192.)"""
    err_exact, err_frozen = _pair_errors(oracle, 6, 0.05, 0, (64, 128, 256))
    assert np.all(err_exact < 0.1 * err_frozen), (err_exact, err_frozen)


def test_sweep_exact_schedule_and_limits(oracle):
    """batch_sites = 1: identical to the sequential oracle sweep, bit for bit.  batch_sites > 1: a hand-rolled Algorithm 1 loop
    around exact_batch_dS; and closer to the sequential chain's Delta S than the frozen sweep is (Lorentz kernel, the paper's)."""
    cfg = wl.CONFIGS[1]
    L, M, K = cfg.L, 64, 128
    S, prop, uni = wl.make_workload(cfg, n_sweeps=1)
    seq = oracle.sweep(L, cfg.t, cfg.JH, cfg.T, 0.0, M, K, 1, 4.0, S, 1, 1, prop, uni)
    ex1 = oracle.sweep_exact(L, cfg.t, cfg.JH, cfg.T, 0.0, M, K, 1, 4.0, S, 1, 1, prop, uni)
    for k in ("dS", "accept", "spins", "magnetization", "n_accepted"):
        assert np.array_equal(seq[k], ex1[k]), k
    Bs = 8
    ex = oracle.sweep_exact(L, cfg.t, cfg.JH, cfg.T, 0.0, M, K, 1, 4.0, S, 1, Bs, prop, uni, nthreads=2)
    Sc = S.copy()
    for colour in (0, 1):
        order = wl.colour_sites(L, colour)
        for st in range(0, len(order), Bs):
            b = order[st:st + Bs]
            dS, acc = oracle.exact_batch_dS(L, cfg.t, cfg.JH, cfg.T, 0.0, M, K, 1, 4.0, Sc, b, prop[0][b], uni[0][b])
            assert np.array_equal(ex["dS"][0][b], dS) and np.array_equal(ex["accept"][0][b], acc)
            Sc[b[acc == 1]] = prop[0][b[acc == 1]]
    assert np.array_equal(ex["spins"], Sc)
    assert ex["n_accepted"][0] == ex["accept"].sum() and abs(ex["magnetization"][0] - oracle.magnetization(Sc)) < 1e-15
    # as long as the decisions agree with the sequential chain the configurations agree, and Delta S must be close to it
    fr = oracle.sweep(L, cfg.t, cfg.JH, cfg.T, 0.0, M, K, 1, 4.0, S, 1, Bs, prop, uni)
    first = wl.colour_sites(L, 0)[:Bs]
    assert np.array_equal(ex["accept"][0][first], seq["accept"][0][first])
    e_exact = np.abs(ex["dS"][0][first] - seq["dS"][0][first]).max()
    e_frozen = np.abs(fr["dS"][0][first] - seq["dS"][0][first]).max()
    assert e_exact < 0.2 * e_frozen, (e_exact, e_frozen)
