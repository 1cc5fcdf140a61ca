/*
 * gfmc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct fp64 CPU implementation of the hot path of the
 * O(N) Green-function-based Monte Carlo (GFMC) method of arXiv:1303.6016 for the
 * 3D double-exchange model, written from the paper (citations are PAPER.md lines).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or constant with the CUDA path (paper_1303_6016_b200/csrc).
 *
 * The method is an approximation + an iteration (a truncated, kernel-damped
 * Chebyshev series inside a Monte Carlo chain), so the oracle follows the
 * algorithm step by step in the paper's order: no moment doubling (Eq. 27-28 are
 * NOT used here: every moment is the direct read-out of Eq. 25-26), no batching,
 * no blocking, no fusion.  Readings of silent/garbled passages are the ones listed
 * in DESIGN.md ("Readings of the paper") and SURVEY.md section 8(c).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): dense diagonalisation for
 * L <= 4, closed-form moments (mu_0..mu_2, ferromagnet band, Neel state),
 * invariants (Hermiticity, |mu|<=1, trace identity, SU(2) covariance), the
 * Chebyshev generating function for the Green-function series, the eigenvalue
 * product formula Eq. (12) for d(z) and its phase, a closed-form integral for the
 * quadrature, exact Delta S_eff from Eq. (7) at large M, and a hand-rolled
 * Algorithm-1 loop for the sweep schedule.  No function below is "parity unpinned".
 *
 * Conventions: site i = x + L*(y + L*z); row = 2*i + sigma (sigma = 0 up, 1 down);
 * complex numbers are C99 `double complex` (interleaved re, im).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define ORACLE_PI 3.14159265358979323846264338327950288

/* ---------------------------------------------------------------- a1: bound
 * The paper requires H~ with spectrum inside [-1,1] but gives no formula
 * (PAPER.md:166, 178).  Reading 9: spin-independent Gershgorin bound.  Row (i,up)
 * of Eq. (1) has centre J_H S^z_i and radius 6|t| + |J_H| sqrt(1-(S^z_i)^2);
 * max over the unit sphere of |S^z| + sqrt(1-S^z^2) is sqrt(2).  b = 0.        */
void gfmc_oracle_bounds(double t, double JH, double *a, double *b)
{
    *a = 6.0 * fabs(t) + sqrt(2.0) * fabs(JH);
    *b = 0.0;
}

/* ---------------------------------------------------------------- O1: operator
 * Eq. (1):  H = -t sum_<ij>,s (c+_is c_js + h.c.)
 *                              + J_H sum_i S_i . c+_ia sigma_ab c_ib,
 * periodic simple-cubic lattice (reading 20), sign of the Hund term as printed
 * (reading 2).  (S.sigma) = [[Sz, Sx - i Sy], [Sx + i Sy, -Sz]].
 * All six directions are always summed (for L = 2 a neighbour counts twice).   */
void gfmc_oracle_apply_H(int L, double t, double JH, const double *S,
                         const cplx *x, cplx *y)
{
    for (int z = 0; z < L; ++z)
    for (int yy = 0; yy < L; ++yy)
    for (int xx = 0; xx < L; ++xx) {
        int i = xx + L * (yy + L * z);
        int nb[6];
        nb[0] = ((xx + 1) % L)     + L * (yy + L * z);
        nb[1] = ((xx + L - 1) % L) + L * (yy + L * z);
        nb[2] = xx + L * (((yy + 1) % L)     + L * z);
        nb[3] = xx + L * (((yy + L - 1) % L) + L * z);
        nb[4] = xx + L * (yy + L * ((z + 1) % L));
        nb[5] = xx + L * (yy + L * ((z + L - 1) % L));
        cplx hop_up = 0.0, hop_dn = 0.0;
        for (int d = 0; d < 6; ++d) {
            hop_up += x[2 * nb[d] + 0];
            hop_dn += x[2 * nb[d] + 1];
        }
        double Sx = S[3 * i + 0], Sy = S[3 * i + 1], Sz = S[3 * i + 2];
        cplx xu = x[2 * i + 0], xd = x[2 * i + 1];
        cplx hund_up = Sz * xu + (Sx - I * Sy) * xd;
        cplx hund_dn = (Sx + I * Sy) * xu - Sz * xd;
        y[2 * i + 0] = -t * hop_up + JH * hund_up;
        y[2 * i + 1] = -t * hop_dn + JH * hund_dn;
    }
}

/* ---------------------------------------------------------------- O2: moments
 * Eq. (25)-(26):  |a_0> = |o beta>, |a_1> = H~|a_0>,
 * |a_m> = 2 H~ |a_{m-1}> - |a_{m-2}>,  mu_m(alpha,beta) = <o alpha|a_m>.
 * mu is [M][2][2] (alpha, beta) complex.  M-1 applications of H per start
 * vector; the doubling of Eq. (27)-(28) is deliberately not used.             */
int gfmc_oracle_moments(int L, double t, double JH, const double *S,
                        int site, int M, cplx *mu)
{
    int N = L * L * L, D = 2 * N;
    double a, b;
    gfmc_oracle_bounds(t, JH, &a, &b);
    if (site < 0 || site >= N || M < 1) return -1;
    cplx *r0 = malloc(sizeof(cplx) * D), *r1 = malloc(sizeof(cplx) * D),
         *hx = malloc(sizeof(cplx) * D);
    if (!r0 || !r1 || !hx) { free(r0); free(r1); free(hx); return -2; }
    for (int beta = 0; beta < 2; ++beta) {
        memset(r0, 0, sizeof(cplx) * D);
        r0[2 * site + beta] = 1.0;                       /* |a_0> = |o beta> */
        for (int al = 0; al < 2; ++al) mu[(0 * 2 + al) * 2 + beta] = r0[2 * site + al];
        if (M > 1) {
            gfmc_oracle_apply_H(L, t, JH, S, r0, hx);
            for (int j = 0; j < D; ++j) r1[j] = (hx[j] - b * r0[j]) / a;   /* |a_1> = H~|a_0> */
            for (int al = 0; al < 2; ++al) mu[(1 * 2 + al) * 2 + beta] = r1[2 * site + al];
        }
        for (int m = 2; m < M; ++m) {
            gfmc_oracle_apply_H(L, t, JH, S, r1, hx);
            for (int j = 0; j < D; ++j) {
                cplx nxt = 2.0 * ((hx[j] - b * r1[j]) / a) - r0[j];       /* Eq. (26) */
                r0[j] = r1[j];
                r1[j] = nxt;
            }
            for (int al = 0; al < 2; ++al) mu[(m * 2 + al) * 2 + beta] = r1[2 * site + al];
        }
    }
    free(r0); free(r1); free(hx);
    return 0;
}

/* Same recursion for many sites; OpenMP over sites is used ONLY by the timed CPU
 * baseline (bench.py cpu_baseline / --impl reference).  mu is [n][M][2][2].    */
int gfmc_oracle_moments_many(int L, double t, double JH, const double *S,
                             const int32_t *sites, int n, int M, cplx *mu, int nthreads)
{
    int rc = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int s = 0; s < n; ++s) {
        int r = gfmc_oracle_moments(L, t, JH, S, sites[s], M, mu + (size_t)s * M * 4);
        if (r != 0) {
#ifdef _OPENMP
#pragma omp critical
#endif
            rc = r;
        }
    }
    return rc;
}

/* ---------------------------------------------------------------- a4: kernel
 * g_m "to eliminate Gibbs oscillations".  kernel 0 = Jackson
 * (BASELINE.json; reading 8):
 *   g_m = [(M-m+1) cos(pi m/(M+1)) + sin(pi m/(M+1)) cot(pi/(M+1))]/(M+1);
 * kernel 1 = Lorentz, the paper's: g_m = sinh[lambda(1-m/M)]/sinh(lambda);
 * kernel 2 = none (g_m = 1).                                                   */
int gfmc_oracle_kernel(int kernel, int M, double lambda, double *g)
{
    for (int m = 0; m < M; ++m) {
        if (kernel == 0) {
            double q = ORACLE_PI / (M + 1.0);
            g[m] = ((M - m + 1.0) * cos(q * m) + sin(q * m) / tan(q)) / (M + 1.0);
        } else if (kernel == 1) {
            g[m] = sinh(lambda * (1.0 - (double)m / M)) / sinh(lambda);
        } else if (kernel == 2) {
            g[m] = 1.0;
        } else return -1;
    }
    return 0;
}

/* ---------------------------------------------------------------- a5: G on the grid
 * Second line of Eq. (24) (reading 7), on the Chebyshev nodes of PAPER.md:193
 * with K points (reading 10), in the form of Eq. (29)-(30), PAPER.md:197-201:
 *   phi_k = pi (k+1/2)/K,  x_k = cos phi_k,  E_k = a x_k + b,
 *   G~_ab(x_k) = (2i / sin phi_k) sum_{m=0}^{M-1} mu'_m(a,b) exp(-i m phi_k),
 *   mu'_0 = g_0 mu_0 / 2,  mu'_m = g_m mu_m.
 * The series is linear in the moments, so the complex off-diagonal moments
 * <o up|T_m|o dn> give G_{up,dn} directly (the paper's Eq. 33-36 detour is not
 * needed on the Eq. (1) path).  Twiddles use the exact integer reduction
 * p = m (2k+1) mod 4K, angle = pi p / (2K).  Gt is G~ [K][2][2]; physical
 * G = G~/a.  E is [K] physical energies (descending).                          */
int gfmc_oracle_green(int M, int K, const cplx *mu, int kernel, double lambda,
                      double a, double b, double *E, cplx *Gt)
{
    double *g = malloc(sizeof(double) * M);
    if (!g) return -2;
    if (gfmc_oracle_kernel(kernel, M, lambda, g) != 0) { free(g); return -1; }
    for (int k = 0; k < K; ++k) {
        double phi = ORACLE_PI * (k + 0.5) / K;
        if (E) E[k] = a * cos(phi) + b;
        cplx acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (int m = 0; m < M; ++m) {
            int64_t p = ((int64_t)m * (2 * k + 1)) % (4 * (int64_t)K);
            double ang = ORACLE_PI * (double)p / (2.0 * K);
            cplx tw = cos(ang) - I * sin(ang);                 /* exp(-i m phi_k) */
            double w = (m == 0) ? 0.5 * g[0] : g[m];           /* Eq. (30) */
            for (int e = 0; e < 4; ++e) acc[e] += w * mu[m * 4 + e] * tw;
        }
        cplx pref = 2.0 * I / sin(phi);
        for (int e = 0; e < 4; ++e) Gt[k * 4 + e] = pref * acc[e];
    }
    free(g);
    return 0;
}

/* overflow-safe Fermi function 1/(1+exp(beta(E-mu))) of Eq. (14) */
static double fermi(double E, double beta, double mu_chem)
{
    double x = beta * (E - mu_chem);
    if (x > 0.0) { double e = exp(-x); return e / (1.0 + e); }
    return 1.0 / (1.0 + exp(x));
}

/* ---------------------------------------------------------------- a6: Delta S_eff
 * Single-site change S_o -> S'_o in Eq. (1):  Delta = H' - H (reading 16) is the
 * 2x2 on-site block J_H (S'-S).sigma, so Eq. (11) d(z) = Det[1 + G(z) Delta]
 * reduces, by the same argument as Eq. (17)-(22),
 * to the 2x2 determinant det(1_2 + G_oo(z) Delta_o) in the basis {o up, o dn}.
 * Eq. (14):  Delta S = (beta/pi) Int f(E) Im log d(E+i0) dE.
 *   Delta~ = (J_H/a) (S'-S).sigma;  A_k = G~(x_k) Delta~;
 *   d_k = (1+A_uu)(1+A_dd) - A_ud A_du;
 *   continuous phase from the top of the band (reading 11):
 *     theta_0 = Arg d_0, theta_k = theta_{k-1} + Arg(d_k conj d_{k-1});
 *   Gauss-Chebyshev midpoint rule (reading 10):
 *     Delta S = (beta a / K) sum_k f(E_k) theta_k sin phi_k.
 * theta_out (optional) receives theta_k; d_out (optional) receives d_k.         */
double gfmc_oracle_delta_S(int K, const cplx *Gt, const double *S_old, const double *S_new,
                           double JH, double a, double b, double T, double mu_chem,
                           double *theta_out, cplx *d_out)
{
    double beta = 1.0 / T;
    double dx = S_new[0] - S_old[0], dy = S_new[1] - S_old[1], dz = S_new[2] - S_old[2];
    double c = JH / a;
    cplx D00 = c * dz, D01 = c * (dx - I * dy), D10 = c * (dx + I * dy), D11 = -c * dz;
    double sum = 0.0, theta = 0.0;
    cplx dprev = 1.0;
    for (int k = 0; k < K; ++k) {
        const cplx *G = Gt + 4 * k;       /* G[0]=uu, G[1]=ud, G[2]=du, G[3]=dd */
        cplx A00 = G[0] * D00 + G[1] * D10;
        cplx A01 = G[0] * D01 + G[1] * D11;
        cplx A10 = G[2] * D00 + G[3] * D10;
        cplx A11 = G[2] * D01 + G[3] * D11;
        cplx d = (1.0 + A00) * (1.0 + A11) - A01 * A10;
        if (k == 0) theta = carg(d);
        else        theta += carg(d * conj(dprev));
        dprev = d;
        if (theta_out) theta_out[k] = theta;
        if (d_out) d_out[k] = d;
        double phi = ORACLE_PI * (k + 0.5) / K;
        double E = a * cos(phi) + b;
        sum += fermi(E, beta, mu_chem) * theta * sin(phi);
    }
    return beta * a / K * sum;
}

/* ---------------------------------------------------------------- a8: magnetization
 * Algorithm 1 line 15: |sum_i S_i| / N.                           */
double gfmc_oracle_magnetization(int N, const double *S)
{
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int i = 0; i < N; ++i) { sx += S[3 * i]; sy += S[3 * i + 1]; sz += S[3 * i + 2]; }
    return sqrt(sx * sx + sy * sy + sz * sz) / N;
}

/* Delta S for one site against the configuration S (moments -> G -> Delta S). */
int gfmc_oracle_site_dS(int L, double t, double JH, double T, double mu_chem,
                        int M, int K, int kernel, double lambda,
                        const double *S, int site, const double *S_new, double *dS)
{
    double a, b;
    gfmc_oracle_bounds(t, JH, &a, &b);
    cplx *mu = malloc(sizeof(cplx) * M * 4), *Gt = malloc(sizeof(cplx) * K * 4);
    if (!mu || !Gt) { free(mu); free(Gt); return -2; }
    int rc = gfmc_oracle_moments(L, t, JH, S, site, M, mu);
    if (rc == 0) rc = gfmc_oracle_green(M, K, mu, kernel, lambda, a, b, NULL, Gt);
    if (rc == 0) *dS = gfmc_oracle_delta_S(K, Gt, S + 3 * site, S_new, JH, a, b, T, mu_chem, NULL, NULL);
    free(mu); free(Gt);
    return rc;
}

/* ---------------------------------------------------------------- O5: sweep
 * Algorithm 1, with BASELINE.json's batching ("frozen batch",
 * DESIGN.md): colour c(i) = (x+y+z) mod 2; for each sweep, for c in (0,1), the
 * sites of colour c in increasing index order are cut into consecutive batches of
 * batch_sites; every site of a batch is evaluated against the SAME configuration
 * (the one at batch start) with proposals[s][i]; accept iff -Delta S > ln u
 * (line 10; reading 15); then all accepted flips are applied
 * (line 11-12; matrix-free, so "update H" is the spin write).  After both
 * colours: magnetization (line 15).  batch_sites = 1 is the paper's strictly
 * sequential algorithm with a deterministic site order (reading 14).
 * S is updated in place.  dS_log/accept_log [n_sweeps][N] (indexed by site) may
 * be NULL.  nthreads > 1 spreads the sites of one batch over OpenMP threads
 * (results are identical: each site is independent inside a batch).            */
int gfmc_oracle_sweep(int L, double t, double JH, double T, double mu_chem,
                      int M, int K, int kernel, double lambda, double *S,
                      int n_sweeps, int batch_sites,
                      const double *proposals, const double *uniforms,
                      double *dS_log, uint8_t *accept_log,
                      double *magnetization, int64_t *n_accepted, int nthreads)
{
    int N = L * L * L;
    if (batch_sites < 1) return -1;
    int *order = malloc(sizeof(int) * N);
    double *dS = malloc(sizeof(double) * N);
    uint8_t *acc = malloc(N);
    if (!order || !dS || !acc) { free(order); free(dS); free(acc); return -2; }
    int rc_all = 0;
    for (int s = 0; s < n_sweeps; ++s) {
        const double *prop = proposals + (size_t)s * N * 3;
        const double *uni = uniforms + (size_t)s * N;
        int64_t nacc = 0;
        for (int colour = 0; colour < 2; ++colour) {
            int n = 0;
            for (int i = 0; i < N; ++i) {
                int x = i % L, y = (i / L) % L, z = i / (L * L);
                if (((x + y + z) & 1) == colour) order[n++] = i;
            }
            for (int start = 0; start < n; start += batch_sites) {
                int cnt = (n - start < batch_sites) ? (n - start) : batch_sites;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1)
#endif
                for (int j = 0; j < cnt; ++j) {
                    int i = order[start + j];
                    double v = 0.0;
                    int rc = gfmc_oracle_site_dS(L, t, JH, T, mu_chem, M, K, kernel, lambda,
                                                 S, i, prop + 3 * i, &v);
                    if (rc != 0) rc_all = rc;
                    dS[j] = v;
                    acc[j] = (-v > log(uni[i])) ? 1 : 0;
                }
                for (int j = 0; j < cnt; ++j) {
                    int i = order[start + j];
                    if (dS_log) dS_log[(size_t)s * N + i] = dS[j];
                    if (accept_log) accept_log[(size_t)s * N + i] = acc[j];
                    if (acc[j]) {
                        S[3 * i] = prop[3 * i]; S[3 * i + 1] = prop[3 * i + 1]; S[3 * i + 2] = prop[3 * i + 2];
                        ++nacc;
                    }
                }
            }
        }
        if (magnetization) magnetization[s] = gfmc_oracle_magnetization(N, S);
        if (n_accepted) n_accepted[s] = nacc;
    }
    free(order); free(dS); free(acc);
    return rc_all;
}
