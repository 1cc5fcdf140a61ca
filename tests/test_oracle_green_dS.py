"""Pins for the oracle's kernel damping (a4), Green-function series (a5/O3), d(z), phase
unwrap, quadrature and Delta S_eff (a6/O4), and the sweep schedule (O5).  No CUDA here."""
import numpy as np
import pytest

from paper_1303_6016_b200 import workload as wl
from tests.dense import SIGMA, dense_H


def _a(t, JH):
    return 6 * abs(t) + np.sqrt(2.0) * abs(JH)


# ------------------------------------------------------------------ a4 kernels
def test_jackson_kernel_textbook_properties(oracle):
    for M in (8, 64, 257):
        g = oracle.kernel(0, M)
        assert g[0] == pytest.approx(1.0, abs=1e-15)
        assert g[1] == pytest.approx(np.cos(np.pi / (M + 1)), abs=1e-14)     # g_1 = cos(pi/(M+1))
        assert np.all(np.diff(g) < 0) and np.all(g > 0)
        # the formula continued to m = M vanishes: last kept coefficient is O(1/M^2)
        assert g[-1] < 10.0 / M ** 2 * np.pi ** 2


def test_jackson_kernel_positive_delta(oracle):
    """Jackson damping of the delta-function series is non-negative (Fejer-like kernel):
    sum_m (2 - delta_m0) g_m T_m(x0) T_m(x) >= 0 for all x."""
    M = 32
    g = oracle.kernel(0, M)
    x = np.cos(np.pi * (np.arange(400) + 0.5) / 400)
    for x0 in (-0.83, 0.0, 0.41):
        s = sum((2 - (m == 0)) * g[m] * np.cos(m * np.arccos(x0)) * np.cos(m * np.arccos(x)) for m in range(M))
        assert s.min() > -1e-12


def test_lorentz_and_none_kernels(oracle):
    M, lam = 50, 4.0
    g = oracle.kernel(1, M, lam)
    m = np.arange(M)
    assert np.allclose(g, np.sinh(lam * (1 - m / M)) / np.sinh(lam), rtol=0, atol=1e-15)
    assert g[0] == 1.0
    assert np.array_equal(oracle.kernel(2, M), np.ones(M))


# ------------------------------------------------------------------ a5 series
def test_green_series_against_chebyshev_generating_function(oracle):
    """Feed mu_m = T_m(eps) e^{-m eta} (kernel 'none', M so large that e^{-M eta} ~ 0).  Then
    sum_m T_m(eps) w^m = (1 - w eps)/(1 - 2 w eps + w^2), w = exp(-i phi'), phi' = phi - i eta, gives
    G~(x_k) = [sin phi' / sin phi] / (eps - cos phi') = resolvent 1/(eps - z) at z = cos(phi - i eta):
    pins the sign of the exponent, the 2i/sin(phi) prefactor, the mu_0/2 of Eq. (30), the node
    grid and the element order of the 2x2 block."""
    M, K = 1500, 37
    eps = np.array([[0.31, -0.72], [0.05, 0.9]])
    eta = np.array([[0.03, 0.05], [0.04, 0.06]])
    m = np.arange(M)[:, None, None]
    mu = np.cos(m * np.arccos(eps)) * np.exp(-m * eta)
    a, b = 3.0, 0.25
    E, Gt = oracle.green(mu, K, 2, 0.0, a, b)
    phi = np.pi * (np.arange(K) + 0.5) / K
    assert np.allclose(E, a * np.cos(phi) + b, rtol=0, atol=1e-14)
    assert np.all(np.diff(E) < 0)
    phic = phi[:, None, None] - 1j * eta[None]
    ref = np.sin(phic) / np.sin(phi)[:, None, None] / (eps[None] - np.cos(phic))
    assert np.abs(Gt - ref).max() < 2e-12 * np.abs(ref).max()
    assert np.all(Gt.imag > 0)                    # Im 1/(eps - z) > 0 for Im z > 0 (G = 1/(H - z), Eq. (10))


def test_green_sum_rule(oracle):
    """(1/K) sum_k sin(phi_k) Im G~_aa(x_k) = g_0 mu_0 = 1 for M <= 2K."""
    L, t, JH, M = 3, 1.0, 4.0, 40
    S = wl.make_spins(L, seed=2)
    mu = oracle.moments(L, t, JH, S, 4, M)
    for kind in (0, 1, 2):
        for K in (M // 2, M, 2 * M, 3 * M + 1):
            _, Gt = oracle.green(mu, K, kind, 4.0, _a(t, JH), 0.0)
            phi = np.pi * (np.arange(K) + 0.5) / K
            for al in range(2):
                assert np.mean(np.sin(phi) * Gt[:, al, al].imag) == pytest.approx(1.0, abs=1e-12)


def test_green_lorentz_close_to_exact_resolvent(oracle):
    """Lorentz damping g_m = sinh[lambda(1-m/M)]/sinh(lambda) = e^{-m lambda/M} (1 + O(e^{-2 lambda(1-m/M)})), so the damped
    series of the TRUE moments approaches [sin phi'/sin phi] <o a|1/(H~ - z)|o b> at z = cos(phi'), phi' = phi - i lambda/M,
    up to O(e^{-2 lambda}): sign and normalisation of the whole chain moments -> G against the dense resolvent."""
    L, t, JH, M = 4, 1.0, 4.0, 512
    S = wl.make_spins(L, seed=1)
    a = _a(t, JH)
    e, V = np.linalg.eigh(dense_H(L, t, JH, S))
    site, K = 11, 64
    mu = oracle.moments(L, t, JH, S, site, M)
    phi = np.pi * (np.arange(K) + 0.5) / K
    rows = V[2 * site:2 * site + 2, :]
    for lam, tol in ((4.0, 0.05), (8.0, 1e-3)):
        _, Gt = oracle.green(mu, K, 1, lam, a, 0.0)
        worst = 0.0
        for k in range(K):
            phic = phi[k] - 1j * lam / M
            Gex = (rows / (e / a - np.cos(phic))[None, :]) @ rows.conj().T * np.sin(phic) / np.sin(phi[k])
            worst = max(worst, np.abs(Gt[k] - Gex).max() / np.abs(Gex).max())
        assert worst < tol, (lam, worst)


# ------------------------------------------------------------------ a6 d(z), phase, quadrature
def _exact_block_G(e, V, site, z):
    rows = V[2 * site:2 * site + 2, :]
    return (rows / (e - z)[None, :]) @ rows.conj().T


def test_d_and_phase_against_eigenvalue_product(oracle):
    """Eq. (11)-(12): det(1 + G(z) Delta) = prod(eps'_i - z)/prod(eps_i - z); the unwrapped phase equals
    sum_i Arg(eps'_i - z) - sum_i Arg(eps_i - z) (each term continuous in E for Im z = eta > 0)."""
    L, t, JH, T = 3, 1.0, 4.0, 0.3
    a = _a(t, JH)
    S = wl.make_spins(L, seed=6)
    site = 7
    Snew = -S[site]
    S2 = S.copy(); S2[site] = Snew
    e, V = np.linalg.eigh(dense_H(L, t, JH, S))
    e2 = np.linalg.eigvalsh(dense_H(L, t, JH, S2))
    K, eta = 2000, 0.01
    phi = np.pi * (np.arange(K) + 0.5) / K
    E = a * np.cos(phi)
    Gt = np.stack([a * _exact_block_G(e, V, site, Ek + 1j * eta) for Ek in E])
    _, theta, d = oracle.delta_S(Gt, S[site], Snew, JH, a, 0.0, T, 0.0, want_theta=True)
    z = E + 1j * eta
    dref = np.prod((e2[None, :] - z[:, None]) / (e[None, :] - z[:, None]), axis=1)
    assert np.abs(d - dref).max() < 1e-11 * np.abs(dref).max()
    thref = (np.angle(e2[None, :] - z[:, None]) - np.angle(e[None, :] - z[:, None])).sum(axis=1)
    assert np.abs(theta - thref).max() < 1e-10
    assert np.abs(theta).max() > 2.9          # close to the +-pi edge of the principal branch


def test_phase_is_continued_beyond_the_principal_branch(oracle):
    """Reading 11: theta_k = theta_{k-1} + Arg(d_k conj d_{k-1}) from the top of the band.  Synthetic
    G~_k = g_k 1_2 with Delta~ = q sigma_z gives d_k = 1 - (g_k q)^2; choose g_k so that d_k = r_k e^{i th_k}
    with th_k running smoothly from 0.2 to 7.5 (more than one full turn)."""
    K, JH, a = 400, 3.0, 6.0
    q = JH / a * 2.0
    th = np.linspace(0.2, 7.5, K)
    r = 1.0 + 0.3 * np.sin(np.arange(K) * 0.1)
    g = np.sqrt(1 - r * np.exp(1j * th) + 0j) / q
    Gt = g[:, None, None] * np.eye(2)[None]
    _, theta, d = oracle.delta_S(Gt, [0, 0, -1.0], [0, 0, 1.0], JH, a, 0.0, 1.0, 0.0, want_theta=True)
    assert np.abs(d - r * np.exp(1j * th)).max() < 1e-13
    assert np.abs(theta - th).max() < 1e-12


def test_quadrature_against_closed_form_integral(oracle):
    """With f == 1 (mu_chem far above the band) Delta S = (beta/pi) int_{-a}^{a} theta(E) dE, and
    theta(E) = sum_i [atan((eps'_i - E)/eta) - atan((eps_i - E)/eta)] integrates in closed form."""
    L, t, JH, T = 3, 1.0, 4.0, 0.7
    a = _a(t, JH)
    S = wl.make_spins(L, seed=8)
    site = 20
    Snew = np.array([0.0, 0.6, -0.8])
    S2 = S.copy(); S2[site] = Snew
    e, V = np.linalg.eigh(dense_H(L, t, JH, S))
    e2 = np.linalg.eigvalsh(dense_H(L, t, JH, S2))
    K, eta = 8192, 0.8
    phi = np.pi * (np.arange(K) + 0.5) / K
    E = a * np.cos(phi)
    Gt = np.stack([a * _exact_block_G(e, V, site, Ek + 1j * eta) for Ek in E])
    val = oracle.delta_S(Gt, S[site], Snew, JH, a, 0.0, T, 1e9)

    def F(u):                                   # antiderivative of atan
        return u * np.arctan(u) - 0.5 * np.log1p(u * u)

    def integral(eps):                          # int_{-a}^{a} atan((eps - E)/eta) dE
        return eta * (F((eps + a) / eta) - F((eps - a) / eta))

    ref = (1.0 / T) / np.pi * (integral(e2).sum() - integral(e).sum())
    assert val == pytest.approx(ref, rel=2e-6)


def test_fermi_weight(oracle):
    """theta == const pins the Fermi factor: (beta a/K) sum f(E_k) sin(phi_k) theta0 -> (beta/pi) theta0 *
    pi * int f dE... checked against the closed form int_{-a}^{a} f(E) dE = a - T ln[(1+e^{(a-mu)/T})/(1+e^{(-a-mu)/T})] + ... ."""
    # d(z) = const = e^{i theta0}: realised by G~ = c * 1_2, Delta~ = diag(dz,-dz)*c' -> choose G so det is a pure phase.
    a, T, mu_c, K = 5.0, 0.4, 0.7, 20000
    theta0 = 0.9
    # S' - S = (0,0,2) (flip from -z to +z); Delta~ = (JH/a) * 2 * sigma_z =: q sigma_z.
    JH = 2.5
    q = JH / a * 2.0
    # want (1 + g q)(1 - g q) = e^{i theta0}  ->  g = sqrt(1 - e^{i theta0})/q with G~ = g * 1_2
    g = np.sqrt(1 - np.exp(1j * theta0) + 0j) / q
    Gt = np.tile((g * np.eye(2))[None], (K, 1, 1))
    val = oracle.delta_S(Gt, [0, 0, -1.0], [0, 0, 1.0], JH, a, 0.0, T, mu_c)
    # int_{-a}^{a} dE / (1 + e^{(E-mu)/T}) = [E - T ln(1 + e^{(E-mu)/T})]_{-a}^{a}
    prim = lambda E: E - T * np.logaddexp(0.0, (E - mu_c) / T)
    ref = (1.0 / T) / np.pi * theta0 * (prim(a) - prim(-a))
    assert val == pytest.approx(ref, rel=1e-6)


def test_no_change_gives_zero(oracle):
    L, t, JH = 3, 1.0, 4.0
    S = wl.make_spins(L, seed=9)
    v = oracle.site_dS(L, t, JH, 0.05, 0.0, 32, 64, 0, 4.0, S, 5, S[5])
    assert v == 0.0


def test_delta_S_sign_and_normalisation_vs_exact(oracle):
    """Loose pin (convergence in M is slow and non-monotonic on a tiny discrete spectrum):
    KPM Delta S (Jackson, K = 2M) for full spin reversals against the exact
    -sum_k [log(1+e^{-beta(eps'_k-mu)}) - log(1+e^{-beta(eps_k-mu)})] of Eq. (7), (9).
    A wrong sign, a missing factor 2, pi, a or beta anywhere in a4-a6 fails it."""
    L, t, JH, T = 4, 1.0, 4.0, 0.5
    S = wl.make_spins(L, seed=1)
    for site in (3, 40, 17):
        Snew = -S[site]
        S2 = S.copy(); S2[site] = Snew
        e = np.linalg.eigvalsh(dense_H(L, t, JH, S))
        e2 = np.linalg.eigvalsh(dense_H(L, t, JH, S2))
        exact = -(np.logaddexp(0, -e2 / T).sum() - np.logaddexp(0, -e / T).sum())
        for M in (1024, 4096):
            kpm = oracle.site_dS(L, t, JH, T, 0.0, M, 2 * M, 0, 4.0, S, site, Snew)
            assert abs(kpm - exact) < 0.10 * abs(exact), (site, M, kpm, exact)


# ------------------------------------------------------------------ a8 / O5
def test_magnetization(oracle):
    assert oracle.magnetization(wl.ferromagnet(3, (1, 1, 0))) == pytest.approx(1.0, abs=1e-15)
    assert oracle.magnetization(wl.neel(4)) == 0.0
    S = wl.make_spins(3, seed=1)
    assert oracle.magnetization(S) == pytest.approx(np.linalg.norm(S.sum(0)) / 27, abs=1e-15)


def _hand_rolled_sweeps(oracle, cfgd, S, n_sweeps, B, prop, uni):
    """Algorithm 1 with the colour-major frozen-batch schedule, in Python."""
    L = cfgd["L"]; N = L ** 3
    S = S.copy()
    dS = np.zeros((n_sweeps, N)); acc = np.zeros((n_sweeps, N), dtype=np.uint8)
    mags, naccs = [], []
    for s in range(n_sweeps):
        nacc = 0
        for colour in (0, 1):
            sites = [i for i in range(N) if ((i % L) + ((i // L) % L) + (i // (L * L))) % 2 == colour]
            for st in range(0, len(sites), B):
                batch = sites[st:st + B]
                frozen = S.copy()
                for i in batch:
                    v = oracle.site_dS(L, cfgd["t"], cfgd["JH"], cfgd["T"], 0.0, cfgd["M"], cfgd["K"], 0, 4.0,
                                       frozen, i, prop[s, i])
                    dS[s, i] = v
                    if -v > np.log(uni[s, i]):
                        acc[s, i] = 1; S[i] = prop[s, i]; nacc += 1
        mags.append(np.linalg.norm(S.sum(0)) / N); naccs.append(nacc)
    return S, dS, acc, np.array(mags), np.array(naccs)


@pytest.mark.parametrize("B", [1, 8, 100])
def test_sweep_equals_hand_rolled_algorithm_1(oracle, B):
    cfg = wl.CONFIGS[1]
    cfgd = dict(L=cfg.L, t=cfg.t, JH=cfg.JH, T=cfg.T, M=32, K=64)
    S, prop, uni = wl.make_workload(cfg, n_sweeps=2)
    out = oracle.sweep(cfg.L, cfg.t, cfg.JH, cfg.T, 0.0, 32, 64, 0, 4.0, S, 2, B, prop, uni, nthreads=2)
    S_ref, dS_ref, acc_ref, mag_ref, nacc_ref = _hand_rolled_sweeps(oracle, cfgd, S, 2, B, prop, uni)
    assert np.array_equal(out["dS"], dS_ref)
    assert np.array_equal(out["accept"], acc_ref)
    assert np.array_equal(out["spins"], S_ref)
    assert np.allclose(out["magnetization"], mag_ref, rtol=0, atol=1e-15)
    assert np.array_equal(out["n_accepted"], nacc_ref)
    assert 0 < out["n_accepted"].sum() < 2 * cfg.N


def test_sweep_identity_proposals_always_accepted(oracle):
    cfg = wl.CONFIGS[1]
    S, _, uni = wl.make_workload(cfg, n_sweeps=1)
    out = oracle.sweep(cfg.L, cfg.t, cfg.JH, cfg.T, 0.0, 16, 32, 0, 4.0, S, 1, 4, S[None].copy(), uni)
    assert out["accept"].all() and np.array_equal(out["spins"], S) and np.all(out["dS"] == 0.0)
