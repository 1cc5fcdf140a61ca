"""Pins for the oracle's operator (O1) and moments (O2): SURVEY.md §8(c) "Pins".

Nothing here calls the CUDA path.  The expected values come from dense
diagonalisation (numpy.linalg.eigh), closed forms, or invariants."""
import numpy as np
import pytest

from paper_1303_6016_b200 import workload as wl
from tests.dense import SIGMA, cheb_T, dense_H


def _a(t, JH):
    return 6 * abs(t) + np.sqrt(2.0) * abs(JH)


def test_bounds_closed_form(oracle):
    a, b = oracle.bounds(1.0, 4.0)
    assert a == pytest.approx(11.65685424949238, abs=1e-13) and b == 0.0
    a, b = oracle.bounds(-1.0, -8.0)
    assert a == pytest.approx(17.31370849898476, abs=1e-13)


@pytest.mark.parametrize("L", [2, 3, 4])
def test_apply_H_equals_dense_matvec(oracle, L):
    rng = np.random.default_rng(10 + L)
    S = wl.make_spins(L, seed=100 + L)
    H = dense_H(L, 0.7, 3.1, S)
    assert np.abs(H - H.conj().T).max() == 0.0
    x = rng.standard_normal(2 * L ** 3) + 1j * rng.standard_normal(2 * L ** 3)
    y = oracle.apply_H(L, 0.7, 3.1, S, x)
    assert np.abs(y - H @ x).max() < 1e-13


def test_spectrum_inside_bound(oracle):
    for seed in range(3):
        S = wl.make_spins(4, seed=seed)
        e = np.linalg.eigvalsh(dense_H(4, 1.0, 4.0, S))
        a, _ = oracle.bounds(1.0, 4.0)
        assert np.abs(e).max() < a


@pytest.mark.parametrize("L,JH", [(3, 4.0), (4, 4.0), (4, 8.0)])
def test_moments_vs_dense_diagonalisation(oracle, L, JH):
    """mu_n(a,b) = sum_k <a|k><k|b> T_n(eps_k/a)  (Eq. (25))."""
    t, M = 1.0, 64
    S = wl.make_spins(L, seed=1)
    e, V = np.linalg.eigh(dense_H(L, t, JH, S))
    a = _a(t, JH)
    for site in (0, 5, L ** 3 - 1):
        mu = oracle.moments(L, t, JH, S, site, M)
        rows = V[2 * site:2 * site + 2, :]                       # <o alpha|k>
        for n in range(M):
            ref = (rows * cheb_T(n, e / a)[None, :]) @ rows.conj().T
            assert np.abs(mu[n] - ref).max() < 5e-14, (site, n)


def test_moments_closed_forms_any_configuration(oracle):
    """mu_0 = 1, mu_1 = (J_H/a) S_o.sigma, mu_2 = [2(6t^2+J_H^2)/a^2 - 1] 1 (L >= 3)."""
    L, t, JH = 5, 1.3, 2.7
    S = wl.make_spins(L, seed=7)
    a = _a(t, JH)
    for site in (0, 17, 124):
        mu = oracle.moments(L, t, JH, S, site, 4)
        Ssig = np.einsum("c,cab->ab", S[site], SIGMA)
        assert np.abs(mu[0] - np.eye(2)).max() == 0.0
        assert np.abs(mu[1] - JH / a * Ssig).max() < 1e-15
        assert np.abs(mu[2] - (2 * (6 * t * t + JH * JH) / a ** 2 - 1) * np.eye(2)).max() < 1e-15


def _band_moments(L, t, shift, a, M):
    k = 2 * np.pi * np.arange(L) / L
    eps = -2 * t * (np.cos(k)[:, None, None] + np.cos(k)[None, :, None] + np.cos(k)[None, None, :])
    x = ((eps + shift) / a).ravel()
    return np.array([cheb_T(n, x).mean() for n in range(M)])


@pytest.mark.parametrize("L,nhat", [(4, (0, 0, 1)), (6, (1, 2, -2)), (8, (0.3, -0.5, 0.4))])
def test_ferromagnet_band(oracle, L, nhat):
    """Aligned spins along n: mu_n = mu+_n P+ + mu-_n P-, textbook tight-binding band +- J_H."""
    t, JH, M = 1.0, 4.0, 48
    S = wl.ferromagnet(L, nhat)
    a = _a(t, JH)
    n = S[0]
    nsig = np.einsum("c,cab->ab", n, SIGMA)
    Pp, Pm = (np.eye(2) + nsig) / 2, (np.eye(2) - nsig) / 2
    mp, mm = _band_moments(L, t, +JH, a, M), _band_moments(L, t, -JH, a, M)
    mu = oracle.moments(L, t, JH, S, site=L ** 3 // 3, M=M)
    ref = mp[:, None, None] * Pp + mm[:, None, None] * Pm
    assert np.abs(mu - ref).max() < 5e-14


def test_neel_state(oracle):
    L, t, JH, M = 4, 1.0, 4.0, 40
    S = wl.neel(L)
    a = _a(t, JH)
    k = 2 * np.pi * np.arange(L) / L
    eps = (-2 * t * (np.cos(k)[:, None, None] + np.cos(k)[None, :, None] + np.cos(k)[None, None, :])).ravel()
    Ek = np.sqrt(eps ** 2 + JH ** 2)
    for site, sgn in ((0, +1.0), (1, -1.0)):           # site 0 has S=+z, site 1 has S=-z
        mu = oracle.moments(L, t, JH, S, site, M)
        for n in range(M):
            up = np.mean((1 + sgn * JH / Ek) / 2 * cheb_T(n, Ek / a) + (1 - sgn * JH / Ek) / 2 * cheb_T(n, -Ek / a))
            dn = np.mean((1 - sgn * JH / Ek) / 2 * cheb_T(n, Ek / a) + (1 + sgn * JH / Ek) / 2 * cheb_T(n, -Ek / a))
            assert abs(mu[n, 0, 0] - up) < 5e-14 and abs(mu[n, 1, 1] - dn) < 5e-14
            assert abs(mu[n, 0, 1]) < 1e-15 and abs(mu[n, 1, 0]) < 1e-15


def test_invariants_hermiticity_bound_trace(oracle):
    L, t, JH, M = 3, 1.0, 4.0, 32
    S = wl.make_spins(L, seed=3)
    a = _a(t, JH)
    e = np.linalg.eigvalsh(dense_H(L, t, JH, S))
    mus = oracle.moments_many(L, t, JH, S, np.arange(L ** 3), M)
    assert np.abs(mus).max() <= 1.0 + 1e-14
    assert np.abs(mus - mus.conj().transpose(0, 1, 3, 2)).max() < 1e-14      # mu(b,a) = conj mu(a,b)
    tr = np.einsum("snaa->n", mus)
    ref = np.array([cheb_T(n, e / a).sum() for n in range(M)])
    assert np.abs(tr - ref).max() < 2e-13
    assert np.abs(tr.imag).max() < 1e-13


def test_global_spin_rotation_covariance(oracle):
    """S -> R S  =>  mu_n -> U mu_n U^+ with U = exp(-i gamma/2 u.sigma)."""
    L, t, JH, M = 3, 1.0, 4.0, 24
    S = wl.make_spins(L, seed=4)
    u = np.array([0.2, -0.7, 0.5]); u /= np.linalg.norm(u)
    gamma = 1.234
    Kx = np.array([[0, -u[2], u[1]], [u[2], 0, -u[0]], [-u[1], u[0], 0]])
    R = np.eye(3) + np.sin(gamma) * Kx + (1 - np.cos(gamma)) * Kx @ Kx      # Rodrigues
    usig = np.einsum("c,cab->ab", u, SIGMA)
    U = np.cos(gamma / 2) * np.eye(2) - 1j * np.sin(gamma / 2) * usig
    SR = S @ R.T
    for site in (0, 13):
        mu = oracle.moments(L, t, JH, S, site, M)
        muR = oracle.moments(L, t, JH, SR, site, M)
        assert np.abs(muR - U @ mu @ U.conj().T).max() < 1e-14


def test_moments_many_matches_single_and_threads(oracle):
    L, t, JH, M = 4, 1.0, 4.0, 16
    S = wl.make_spins(L, seed=5)
    sites = np.array([3, 9, 9, 63], dtype=np.int32)
    one = np.stack([oracle.moments(L, t, JH, S, s, M) for s in sites])
    assert np.array_equal(one, oracle.moments_many(L, t, JH, S, sites, M, nthreads=1))
    assert np.array_equal(one, oracle.moments_many(L, t, JH, S, sites, M, nthreads=3))


def test_particle_hole_relations_even_L(oracle):
    """The relations the CUDA path's one-vector mode (ph_symmetry) rests on, checked on the ORACLE's plain
    two-vector recursion: on an even-L periodic lattice A = Gamma (i sigma_y) K gives A H A^-1 = -H for Eq. (1), hence
    mu_n(dn,dn) = (-1)^n mu_n(up,up), mu_even(up,dn) = 0 and mu_odd traceless.  They must FAIL on an odd lattice."""
    M = 24
    for L, ok in ((4, True), (6, True), (3, False), (5, False)):
        S = wl.make_spins(L, seed=70 + L)
        mu = oracle.moments(L, 1.0, 4.0, S, 11, M)
        n = np.arange(M)
        dev = max(np.abs(mu[:, 1, 1] - (-1.0) ** n * mu[:, 0, 0]).max(), np.abs(mu[0::2, 0, 1]).max())
        assert (dev < 1e-13) if ok else (dev > 1e-3), (L, dev)
