"""Pins for the J_H -> infinity oracle (oracle/gfmc_oracle_dex.c): Eq. (2)-(3) operator,
moments in the {o, v} pair of Eq. (21), d(z) of Eq. (22), Delta S_eff and the sweep.  No CUDA here."""
import numpy as np
import pytest

from paper_1303_6016_b200 import workload as wl
from tests.dense import cheb_T, dense_H_dex, spinors


def _rot(axis, ang):
    axis = np.asarray(axis, float) / np.linalg.norm(axis)
    Kx = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + np.sin(ang) * Kx + (1 - np.cos(ang)) * Kx @ Kx


# ------------------------------------------------------------------ Eq. (3)
def test_hopping_equals_spinor_overlap(oracle):
    S = wl.make_spins(4, seed=11)
    chi = spinors(S)
    for i, j in [(0, 1), (5, 9), (17, 3), (40, 41), (2, 2)]:
        tij = oracle.dex_hopping(S[i], S[j])
        assert abs(tij - np.vdot(chi[i], chi[j])) < 1e-14
        assert abs(abs(tij) ** 2 - (1 + S[i] @ S[j]) / 2) < 1e-14          # |t_ij| = cos(Theta_ij / 2)
        assert abs(oracle.dex_hopping(S[j], S[i]) - np.conj(tij)) < 1e-15   # Hermitian bond
    assert oracle.dex_hopping(S[7], S[7]) == pytest.approx(1.0, abs=1e-15)
    assert abs(oracle.dex_hopping([0, 0, 1.0], [0, 0, -1.0])) < 1e-15       # antiparallel spins: no hopping
    assert oracle.dex_bounds(1.5) == (9.0, 0.0)


@pytest.mark.parametrize("L", [3, 4])
def test_apply_H_equals_dense(oracle, L):
    t = 1.3
    S = wl.make_spins(L, seed=20 + L)
    H = dense_H_dex(L, t, S)
    assert np.abs(H - H.conj().T).max() < 1e-15
    rng = np.random.default_rng(5)
    x = rng.standard_normal(L ** 3) + 1j * rng.standard_normal(L ** 3)
    assert np.abs(oracle.dex_apply_H(L, t, S, x) - H @ x).max() < 1e-13
    a, _ = oracle.dex_bounds(t)
    assert np.abs(np.linalg.eigvalsh(H)).max() <= a


def test_v_is_delta_times_o(oracle):
    """Eq. (15), (21): |v> = (H' - H)|o>, and Delta has no other non-zero column but those of o's neighbours."""
    L, t = 4, 0.8
    S = wl.make_spins(L, seed=31)
    site, Snew = 22, wl.make_spins(1, seed=77)[0]
    S2 = S.copy(); S2[site] = Snew
    Delta = dense_H_dex(L, t, S2) - dense_H_dex(L, t, S)
    nb, v = oracle.dex_v(L, t, S, site, Snew)
    col = np.zeros(L ** 3, complex); col[nb] = v
    assert np.abs(col - Delta[:, site]).max() < 1e-14
    rest = Delta.copy(); rest[:, site] = 0; rest[site, :] = 0
    assert np.abs(rest).max() == 0.0
    assert sorted(nb) == sorted(np.flatnonzero(np.abs(dense_H_dex(L, 1.0, wl.ferromagnet(L))[:, site]) > 0))


# ------------------------------------------------------------------ moments
def _eig_moments(H, H2, site, a, M):
    e, V = np.linalg.eigh(H)
    o = np.zeros(H.shape[0], complex); o[site] = 1
    v = (H2 - H) @ o
    B = np.stack([o, v], axis=1)                      # columns |o>, |v>
    C = V.conj().T @ B                                 # <k|beta>
    return np.stack([(C.conj().T * cheb_T(n, e / a)[None, :]) @ C for n in range(M)])


@pytest.mark.parametrize("L,seed", [(3, 2), (4, 3)])
def test_moments_against_dense_eigh(oracle, L, seed):
    t, M = 1.0, 40
    S = wl.make_spins(L, seed=seed)
    site = 5
    Snew = wl.make_spins(1, seed=seed + 50)[0]
    S2 = S.copy(); S2[site] = Snew
    a, _ = oracle.dex_bounds(t)
    ref = _eig_moments(dense_H_dex(L, t, S), dense_H_dex(L, t, S2), site, a, M)
    mu = oracle.dex_moments(L, t, S, site, Snew, M)
    assert np.abs(mu - ref).max() < 2e-13
    assert np.abs(mu[:, 1, 0] - mu[:, 0, 1].conj()).max() < 1e-13       # T_n(H~) is Hermitian
    assert np.abs(mu[:, 0, 0].imag).max() < 1e-14 and np.abs(mu[:, 0, 0]).max() <= 1 + 1e-14


def test_moments_closed_forms(oracle):
    """mu_0 = [[1, 0], [0, <v|v>]]; mu_1(o,o) = 0, mu_1(o,v) = <o|H~|v> = -(t/a) sum_j t_oj v_j;
    mu_2(o,o) = 2 (t/a)^2 sum_j |t_oj|^2 - 1 with |t_oj|^2 = (1 + S_o.S_j)/2.  Any configuration, L >= 4."""
    L, t = 6, 1.0
    S = wl.make_spins(L, seed=8)
    site, Snew = 100, np.array([0.6, 0.0, -0.8])
    a, _ = oracle.dex_bounds(t)
    nb, v = oracle.dex_v(L, t, S, site, Snew)
    mu = oracle.dex_moments(L, t, S, site, Snew, 3)
    chi = spinors(S)
    t_oj = np.array([np.vdot(chi[site], chi[j]) for j in nb])
    assert np.abs(mu[0] - np.array([[1, 0], [0, np.vdot(v, v).real]])).max() < 1e-14
    assert abs(mu[1, 0, 0]) < 1e-15 and abs(mu[1, 1, 1]) < 1e-15
    assert abs(mu[1, 0, 1] - (-(t / a) * (t_oj * v).sum())) < 1e-14
    assert abs(mu[2, 0, 0] - (2 * (t / a) ** 2 * (1 + S[nb] @ S[site]).sum() / 2 - 1)) < 1e-14


@pytest.mark.parametrize("L", [5, 8])
def test_ferromagnet_band(oracle, L):
    """Aligned spins along any n: t_ij = 1, so H is the free cubic-lattice band eps_k = -2t sum cos k (textbook):
    mu_n(o,o) = L^-3 sum_k T_n(eps_k / a)."""
    t, M = 1.0, 48
    S = wl.ferromagnet(L, (0.3, -0.5, 0.81))
    a, _ = oracle.dex_bounds(t)
    k = 2 * np.pi * np.arange(L) / L
    eps = -2 * t * (np.cos(k)[:, None, None] + np.cos(k)[None, :, None] + np.cos(k)[None, None, :]).ravel()
    ref = np.array([cheb_T(n, eps / a).mean() for n in range(M)])
    mu = oracle.dex_moments(L, t, S, 17, S[17], M)
    assert np.abs(mu[:, 0, 0] - ref).max() < 1e-13
    assert np.abs(mu[:, 1, 1]).max() == 0.0                 # S' = S: |v> = 0


# ------------------------------------------------------------------ d(z), phase, Delta S
def _exact_ov_G(H, H2, site, z):
    n = H.shape[0]
    o = np.zeros(n, complex); o[site] = 1
    v = (H2 - H) @ o
    B = np.stack([o, v], axis=1)
    return B.conj().T @ np.linalg.solve(H - z * np.eye(n), B)       # G = 1/(H - z), Eq. (10)


def test_eq22_equals_full_determinant_and_eigenvalue_product(oracle):
    """Eq. (22) fed with the exact resolvent = Det[1 + G Delta] (Eq. (11), full N x N) = prod(eps'-z)/prod(eps-z)
    (Eq. (12)); the oracle's unwrapped phase = sum Arg(eps'-z) - sum Arg(eps-z)."""
    L, t, T = 4, 1.0, 0.3
    S = wl.make_spins(L, seed=13)
    site = 37
    Snew = -S[site]
    S2 = S.copy(); S2[site] = Snew
    H, H2 = dense_H_dex(L, t, S), dense_H_dex(L, t, S2)
    e, e2 = np.linalg.eigvalsh(H), np.linalg.eigvalsh(H2)
    a, _ = oracle.dex_bounds(t)
    K, eta = 1500, 0.02
    phi = np.pi * (np.arange(K) + 0.5) / K
    z = a * np.cos(phi) + 1j * eta
    Gt = np.stack([a * _exact_ov_G(H, H2, site, zk) for zk in z])
    _, theta, d = oracle.dex_delta_S(Gt, a, 0.0, T, 0.0, want_theta=True)
    dref = np.prod((e2[None, :] - z[:, None]) / (e[None, :] - z[:, None]), axis=1)
    assert np.abs(d - dref).max() < 1e-10 * np.abs(dref).max()
    thref = (np.angle(e2[None, :] - z[:, None]) - np.angle(e[None, :] - z[:, None])).sum(axis=1)
    assert np.abs(theta - thref).max() < 1e-9
    for kk in (3, 700):
        full = np.linalg.det(np.eye(L ** 3) + np.linalg.inv(H - z[kk] * np.eye(L ** 3)) @ (H2 - H))
        assert abs(d[kk] - full) < 1e-10 * abs(full)


def test_no_change_gives_zero(oracle):
    S = wl.make_spins(4, seed=9)
    assert oracle.dex_site_dS(4, 1.0, 0.05, 0.0, 32, 64, 0, 4.0, S, 5, S[5]) == 0.0


def test_delta_S_sign_and_normalisation_vs_exact(oracle):
    """Loose pin (slow KPM convergence on a 64-level spectrum): KPM Delta S vs Eq. (7), (9) from exact eigenvalues."""
    L, t, T = 4, 1.0, 0.5
    S = wl.make_spins(L, seed=1)
    for site in (3, 40):
        Snew = -S[site]
        S2 = S.copy(); S2[site] = Snew
        e, e2 = np.linalg.eigvalsh(dense_H_dex(L, t, S)), np.linalg.eigvalsh(dense_H_dex(L, t, S2))
        exact = -(np.logaddexp(0, -e2 / T).sum() - np.logaddexp(0, -e / T).sum())
        for M in (1024, 4096):
            kpm = oracle.dex_site_dS(L, t, T, 0.0, M, 2 * M, 0, 4.0, S, site, Snew)
            assert abs(kpm - exact) < 0.12 * abs(exact) + 0.01, (site, M, kpm, exact)


def test_global_rotation_is_a_gauge_transformation(oracle):
    """Rotating every spin (and the proposal) by the same R changes t_ij only by site phases: |t_ij| and both spectra are
    unchanged, so the exact d(z) and Delta S are invariant.  The truncated series is NOT exactly invariant, because the
    Eq. (3) gauge of S'_o relative to S_o changes |v> by more than a phase (reading f1-3): the two gauges agree
    only to truncation accuracy, and agree better as M grows."""
    L, t, T = 4, 1.0, 0.1
    S = wl.make_spins(L, seed=4)
    site, Snew = 9, wl.make_spins(1, seed=99)[0]
    R = _rot((1.0, 2.0, -0.5), 1.1)
    Sr, Snew_r = S @ R.T, R @ Snew
    H, Hr = dense_H_dex(L, t, S), dense_H_dex(L, t, Sr)
    assert np.abs(np.abs(H) - np.abs(Hr)).max() < 1e-14
    assert np.abs(np.linalg.eigvalsh(H) - np.linalg.eigvalsh(Hr)).max() < 1e-13
    x = np.random.default_rng(3).standard_normal(L ** 3) + 0j
    assert np.abs(oracle.dex_apply_H(L, t, Sr, x) - Hr @ x).max() < 1e-13
    gaps = []
    for M in (64, 1024):
        v0 = oracle.dex_site_dS(L, t, T, 0.0, M, 2 * M, 0, 4.0, S, site, Snew)
        v1 = oracle.dex_site_dS(L, t, T, 0.0, M, 2 * M, 0, 4.0, Sr, site, Snew_r)
        assert abs(v0) > 1e-3 and abs(v1 - v0) < 5e-3 * abs(v0)
        gaps.append(abs(v1 - v0))
    assert gaps[1] < gaps[0]


# ------------------------------------------------------------------ sweep
@pytest.mark.parametrize("B", [1, 7])
def test_sweep_equals_hand_rolled_algorithm_1(oracle, B):
    L, t, T, M, K = 4, 1.0, 0.05, 24, 48
    cfg = wl.CONFIGS[1]
    S, prop, uni = wl.make_workload(cfg, n_sweeps=2)
    out = oracle.dex_sweep(L, t, T, 0.0, M, K, 0, 4.0, S, 2, B, prop, uni, nthreads=2)
    N = L ** 3
    Sc = S.copy()
    dS = np.zeros((2, N)); acc = np.zeros((2, N), dtype=np.uint8)
    for s in range(2):
        for colour in (0, 1):
            sites = [i for i in range(N) if ((i % L) + ((i // L) % L) + (i // (L * L))) % 2 == colour]
            for st in range(0, len(sites), B):
                frozen = Sc.copy()
                for i in sites[st:st + B]:
                    dS[s, i] = oracle.dex_site_dS(L, t, T, 0.0, M, K, 0, 4.0, frozen, i, prop[s, i])
                    if -dS[s, i] > np.log(uni[s, i]):
                        acc[s, i] = 1; Sc[i] = prop[s, i]
    assert np.array_equal(out["dS"], dS) and np.array_equal(out["accept"], acc) and np.array_equal(out["spins"], Sc)
    assert out["magnetization"][-1] == pytest.approx(np.linalg.norm(Sc.sum(0)) / N, abs=1e-15)
    assert 0 < out["n_accepted"].sum() < 2 * N
