/*
 * gfmc_oracle_exact.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Oracle for SURVEY.md section 8(f) row f5, "exactness inside a batch", for the
 * Hamiltonian of Eq. (1), written from the paper; plain C99, fp64,
 * no blocking, no fusion, no doubling.  Same rules as gfmc_oracle.c: only tests/,
 * __graft_entry__.smoke() and bench.py's CPU legs may build, load or call it; it
 * shares no code, header, table or constant with the CUDA path (paper_1303_6016_b200/csrc).
 *
 * What it computes.  The paper's Algorithm 1 is sequential:
 * trial o is evaluated with the Green's function of the CURRENT Hamiltonian, i.e.
 * with every earlier accepted flip applied.  BASELINE.json's batches evaluate all
 * sites of a batch against the configuration at batch start ("frozen batch",
 * gfmc_oracle_sweep).  Here the sites of a batch are processed in order and site
 * B sees the earlier ACCEPTED flips A of the same batch exactly, without a new
 * Chebyshev recursion: with U the set of accepted sites, Delta_U = sum_A Delta_A
 * (each Delta_A = J_H (S'_A - S_A).sigma is a 2x2 on-site block) and
 * G_U(z) = 1/(H + Delta_U - z), Eq. (11) applied to the pair
 * (H + Delta_U, H + Delta_U + Delta_B) gives the exact conditional ratio
 *     d_B|U(z) = Det[1 + G_U(z) Delta_B] = det_2(1_2 + G_U,BB(z) Delta_B)
 * (the same reduction to the touched block as Eq. (17)-(22)),
 * and the resolvent identity G_U = G - G Delta_U G_U restricted to the site
 * blocks (Dyson / Woodbury) gives
 *     G_U,BB = G_BB - G_BU Delta_U (1 + G_UU Delta_U)^-1 G_UB,
 * which needs only the blocks G_XY(z) = <o_X a|G(z)|o_Y b> between the sites of
 * the batch at batch start.  Those come from CROSS moments
 *     mu_m(Xa, Yb) = <o_X a| T_m(H~) |o_Y b> = a_m^{Yb}[Xa]      (Eq. (25)-(26))
 * read out of the very vectors the diagonal moments come from, through the same
 * series Eq. (24)/(29)-(30) (it is linear in the moments; gfmc_oracle_green of
 * gfmc_oracle.c is called block by block).  Delta S, the branch of the phase and
 * the quadrature are those of gfmc_oracle_delta_S (Eq. (14), readings 10-11).
 * The product over the batch of the conditional ratios is the ratio of the joint
 * flip; with the exact resolvent it is exact (pin 1 below), with the truncated,
 * kernel-damped series it agrees with the sequential algorithm up to truncation
 * error (pin 3).
 *
 * Pins (tests/test_oracle_exact.py, `-m "not gpu"`):
 *  1. with the exact resolvent of a dense matrix (L <= 4) at complex z the
 *     conditional d_B|U equals prod(eps'' - z)/prod(eps' - z), eps' / eps'' the
 *     spectra of H + Delta_U and H + Delta_U + Delta_B (Eq. (12)),
 *     and the product of the conditional ratios equals the joint ratio;
 *  2. cross moments against dense eigen-decomposition; mu(X,Y) = mu(Y,X)^dagger;
 *     the diagonal blocks are gfmc_oracle_moments;
 *  3. with KPM moments, a two-site batch reproduces the sequential (batch = 1)
 *     chain's Delta S of the second site to truncation level, shrinking with M,
 *     where the frozen batch does not;
 *  4. no accepted flip, or accepted flips with S' = S, leave every Delta S equal
 *     to the frozen-batch value bit for bit.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define ORACLE_PI 3.14159265358979323846264338327950288

/* from gfmc_oracle.c */
void gfmc_oracle_bounds(double t, double JH, double *a, double *b);
void gfmc_oracle_apply_H(int L, double t, double JH, const double *S, const cplx *x, cplx *y);
int gfmc_oracle_green(int M, int K, const cplx *mu, int kernel, double lambda, double a, double b, double *E, cplx *Gt);
double gfmc_oracle_magnetization(int N, const double *S);

/* ---------------------------------------------------------------- cross moments
 * mu[X][Y][m][al][be] = <o_X al| T_m(H~) |o_Y be>: the plain recursion of
 * Eq. (26) from |o_Y be>, every vector a_m read out at the rows of all n sites
 * (Eq. (25) with <i| replaced by <o_X al|).  OpenMP over start sites Y only.   */
int gfmc_oracle_cross_moments(int L, double t, double JH, const double *S,
                              const int32_t *sites, int n, int M, cplx *mu, int nthreads)
{
    int N = L * L * L, D = 2 * N;
    double a, b;
    gfmc_oracle_bounds(t, JH, &a, &b);
    for (int s = 0; s < n; ++s) if (sites[s] < 0 || sites[s] >= N) return -1;
    if (M < 1) return -1;
    int rc = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int Y = 0; Y < n; ++Y) {
        cplx *r0 = malloc(sizeof(cplx) * D), *r1 = malloc(sizeof(cplx) * D), *hx = malloc(sizeof(cplx) * D);
        if (!r0 || !r1 || !hx) { free(r0); free(r1); free(hx); rc = -2; continue; }
        for (int be = 0; be < 2; ++be) {
#define READ_OUT(vec, m)                                                                        \
            for (int X = 0; X < n; ++X)                                                         \
                for (int al = 0; al < 2; ++al)                                                  \
                    mu[((((size_t)X * n + Y) * M + (m)) * 2 + al) * 2 + be] = (vec)[2 * sites[X] + al];
            memset(r0, 0, sizeof(cplx) * D);
            r0[2 * sites[Y] + be] = 1.0;
            READ_OUT(r0, 0)
            if (M > 1) {
                gfmc_oracle_apply_H(L, t, JH, S, r0, hx);
                for (int j = 0; j < D; ++j) r1[j] = (hx[j] - b * r0[j]) / a;
                READ_OUT(r1, 1)
            }
            for (int m = 2; m < M; ++m) {
                gfmc_oracle_apply_H(L, t, JH, S, r1, hx);
                for (int j = 0; j < D; ++j) {
                    cplx nxt = 2.0 * ((hx[j] - b * r1[j]) / a) - r0[j];
                    r0[j] = r1[j];
                    r1[j] = nxt;
                }
                READ_OUT(r1, m)
            }
#undef READ_OUT
        }
        free(r0); free(r1); free(hx);
    }
    return rc;
}

static double fermi(double E, double beta, double mu_chem)
{
    double x = beta * (E - mu_chem);
    if (x > 0.0) { double e = exp(-x); return e / (1.0 + e); }
    return 1.0 / (1.0 + exp(x));
}

/* solves A Z = B in place (A: m x m, B: m x nrhs, row-major) by Gaussian elimination with partial pivoting */
static int solve_dense(int m, int nrhs, cplx *A, cplx *B)
{
    for (int c = 0; c < m; ++c) {
        int piv = c;
        for (int r = c + 1; r < m; ++r) if (cabs(A[r * m + c]) > cabs(A[piv * m + c])) piv = r;
        if (cabs(A[piv * m + c]) == 0.0) return -3;
        if (piv != c) {
            for (int k = 0; k < m; ++k) { cplx tmp = A[c * m + k]; A[c * m + k] = A[piv * m + k]; A[piv * m + k] = tmp; }
            for (int k = 0; k < nrhs; ++k) { cplx tmp = B[c * nrhs + k]; B[c * nrhs + k] = B[piv * nrhs + k]; B[piv * nrhs + k] = tmp; }
        }
        for (int r = c + 1; r < m; ++r) {
            cplx f = A[r * m + c] / A[c * m + c];
            for (int k = c; k < m; ++k) A[r * m + k] -= f * A[c * m + k];
            for (int k = 0; k < nrhs; ++k) B[r * nrhs + k] -= f * B[c * nrhs + k];
        }
    }
    for (int c = m - 1; c >= 0; --c)
        for (int k = 0; k < nrhs; ++k) {
            cplx v = B[c * nrhs + k];
            for (int j = c + 1; j < m; ++j) v -= A[c * m + j] * B[j * nrhs + k];
            B[c * nrhs + k] = v / A[c * m + c];
        }
    return 0;
}

/* ---------------------------------------------------------------- exact in-batch decisions
 * Gt[X][Y][k][2][2] = G~_XY(x_k) (rescaled, as gfmc_oracle_green returns it) for the n sites of the batch at batch start;
 * S_old / S_new [n][3] current and trial spins, uniforms [n] in (0,1].  Sites are processed in index order 0..n-1:
 *   U = accepted sites so far;  Delta~_A = (J_H/a)(S'_A - S_A).sigma;
 *   G~_U,BB(k) = G~_BB - G~_BU Delta~_U (1 + G~_UU Delta~_U)^-1 G~_UB           (header)
 *   d_k = det_2(1 + G~_U,BB(k) Delta~_B);  Delta S_B by the phase/quadrature of gfmc_oracle_delta_S;
 *   accept iff -Delta S_B > ln u_B  (Alg. 1 line 10).
 * dS [n], accept [n]; d_out (optional) [n][K] receives the conditional d_k.                                            */
int gfmc_oracle_exact_batch(int K, int n, const cplx *Gt, const double *S_old, const double *S_new,
                            const double *uniforms, double JH, double a, double b, double T, double mu_chem,
                            double *dS, uint8_t *accept, cplx *d_out)
{
    double beta = 1.0 / T, c = JH / a;
    int *U = malloc(sizeof(int) * (n > 0 ? n : 1));
    cplx *Dl = malloc(sizeof(cplx) * 4 * (n > 0 ? n : 1));            /* Delta~ of every site, [n][2][2] */
    cplx *A = malloc(sizeof(cplx) * 4 * n * n + 16), *Z = malloc(sizeof(cplx) * 4 * n + 16);
    if (!U || !Dl || !A || !Z) { free(U); free(Dl); free(A); free(Z); return -2; }
    for (int j = 0; j < n; ++j) {
        double dx = S_new[3 * j] - S_old[3 * j], dy = S_new[3 * j + 1] - S_old[3 * j + 1], dz = S_new[3 * j + 2] - S_old[3 * j + 2];
        Dl[4 * j + 0] = c * dz; Dl[4 * j + 1] = c * (dx - I * dy); Dl[4 * j + 2] = c * (dx + I * dy); Dl[4 * j + 3] = -c * dz;
    }
    int nu = 0, rc = 0;
#define GBLK(X, Y, k) (Gt + ((((size_t)(X) * n + (Y)) * K + (k)) * 4))
    for (int B = 0; B < n; ++B) {
        double sum = 0.0, theta = 0.0;
        cplx dprev = 1.0;
        for (int k = 0; k < K; ++k) {
            cplx G[4];
            for (int e = 0; e < 4; ++e) G[e] = GBLK(B, B, k)[e];
            if (nu > 0) {
                int m = 2 * nu;
                /* A = 1 + G~_UU Delta~_U,  Z = G~_UB */
                for (int p = 0; p < nu; ++p) for (int al = 0; al < 2; ++al)
                    for (int q = 0; q < nu; ++q) for (int be = 0; be < 2; ++be) {
                        const cplx *g = GBLK(U[p], U[q], k);
                        cplx v = g[al * 2 + 0] * Dl[4 * U[q] + 0 * 2 + be] + g[al * 2 + 1] * Dl[4 * U[q] + 1 * 2 + be];
                        A[(2 * p + al) * m + (2 * q + be)] = v + ((p == q && al == be) ? 1.0 : 0.0);
                    }
                for (int p = 0; p < nu; ++p) for (int al = 0; al < 2; ++al) for (int be = 0; be < 2; ++be)
                    Z[(2 * p + al) * 2 + be] = GBLK(U[p], B, k)[al * 2 + be];
                if (solve_dense(m, 2, A, Z) != 0) rc = -3;
                /* G~_BB -= sum_q G~_B,Uq Delta~_Uq Z_q */
                for (int q = 0; q < nu; ++q) {
                    const cplx *g = GBLK(B, U[q], k);
                    const cplx *Dq = Dl + 4 * U[q];
                    cplx W[4];                                           /* G~_BUq Delta~_Uq */
                    for (int al = 0; al < 2; ++al) for (int be = 0; be < 2; ++be)
                        W[al * 2 + be] = g[al * 2 + 0] * Dq[0 * 2 + be] + g[al * 2 + 1] * Dq[1 * 2 + be];
                    for (int al = 0; al < 2; ++al) for (int be = 0; be < 2; ++be)
                        G[al * 2 + be] -= W[al * 2 + 0] * Z[(2 * q + 0) * 2 + be] + W[al * 2 + 1] * Z[(2 * q + 1) * 2 + be];
                }
            }
            const cplx *Db = Dl + 4 * B;
            cplx A00 = G[0] * Db[0] + G[1] * Db[2];
            cplx A01 = G[0] * Db[1] + G[1] * Db[3];
            cplx A10 = G[2] * Db[0] + G[3] * Db[2];
            cplx A11 = G[2] * Db[1] + G[3] * Db[3];
            cplx d = (1.0 + A00) * (1.0 + A11) - A01 * A10;
            if (k == 0) theta = carg(d);
            else        theta += carg(d * conj(dprev));
            dprev = d;
            if (d_out) d_out[(size_t)B * K + k] = d;
            double phi = ORACLE_PI * (k + 0.5) / K;
            double E = a * cos(phi) + b;
            sum += fermi(E, beta, mu_chem) * theta * sin(phi);
        }
        dS[B] = beta * a / K * sum;
        accept[B] = (-dS[B] > log(uniforms[B])) ? 1 : 0;
        if (accept[B]) U[nu++] = B;
    }
#undef GBLK
    free(U); free(Dl); free(A); free(Z);
    return rc;
}

/* Delta S and decisions of one batch of sites against the configuration S, exact inside the batch:
 * cross moments -> G~ blocks (gfmc_oracle_green, block by block) -> gfmc_oracle_exact_batch.
 * proposals / uniforms are indexed by position in `sites`.                                                             */
int gfmc_oracle_exact_batch_dS(int L, double t, double JH, double T, double mu_chem, int M, int K, int kernel, double lambda,
                               const double *S, const int32_t *sites, int n, const double *proposals, const double *uniforms,
                               double *dS, uint8_t *accept, int nthreads)
{
    double a, b;
    gfmc_oracle_bounds(t, JH, &a, &b);
    if (n <= 0) return 0;
    cplx *mu = malloc(sizeof(cplx) * (size_t)n * n * M * 4), *Gt = malloc(sizeof(cplx) * (size_t)n * n * K * 4);
    double *So = malloc(sizeof(double) * 3 * n);
    if (!mu || !Gt || !So) { free(mu); free(Gt); free(So); return -2; }
    int rc = gfmc_oracle_cross_moments(L, t, JH, S, sites, n, M, mu, nthreads);
    for (int p = 0; p < n * n && rc == 0; ++p)
        rc = gfmc_oracle_green(M, K, mu + (size_t)p * M * 4, kernel, lambda, a, b, NULL, Gt + (size_t)p * K * 4);
    for (int j = 0; j < n; ++j) for (int cc = 0; cc < 3; ++cc) So[3 * j + cc] = S[3 * sites[j] + cc];
    if (rc == 0) rc = gfmc_oracle_exact_batch(K, n, Gt, So, proposals, uniforms, JH, a, b, T, mu_chem, dS, accept, NULL);
    free(mu); free(Gt); free(So);
    return rc;
}

/* ---------------------------------------------------------------- sweep, exact inside every batch
 * Algorithm 1 with the colour-major batch schedule of gfmc_oracle_sweep, but the sites of a batch are
 * decided one after the other (increasing site index) with gfmc_oracle_exact_batch instead of against the frozen
 * configuration; the accepted flips are written to S after the batch.  batch_sites = 1 is gfmc_oracle_sweep with
 * batch_sites = 1 (the paper's sequential algorithm).                                                                  */
int gfmc_oracle_sweep_exact(int L, double t, double JH, double T, double mu_chem,
                            int M, int K, int kernel, double lambda, double *S,
                            int n_sweeps, int batch_sites,
                            const double *proposals, const double *uniforms,
                            double *dS_log, uint8_t *accept_log,
                            double *magnetization, int64_t *n_accepted, int nthreads)
{
    int N = L * L * L;
    if (batch_sites < 1) return -1;
    int32_t *order = malloc(sizeof(int32_t) * N);
    double *dS = malloc(sizeof(double) * batch_sites), *pr = malloc(sizeof(double) * 3 * batch_sites), *un = malloc(sizeof(double) * batch_sites);
    uint8_t *acc = malloc(batch_sites);
    if (!order || !dS || !pr || !un || !acc) { free(order); free(dS); free(pr); free(un); free(acc); return -2; }
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
                for (int j = 0; j < cnt; ++j) {
                    int i = order[start + j];
                    pr[3 * j] = prop[3 * i]; pr[3 * j + 1] = prop[3 * i + 1]; pr[3 * j + 2] = prop[3 * i + 2];
                    un[j] = uni[i];
                }
                int rc = gfmc_oracle_exact_batch_dS(L, t, JH, T, mu_chem, M, K, kernel, lambda, S, order + start, cnt,
                                                    pr, un, dS, acc, nthreads);
                if (rc != 0) rc_all = rc;
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
    free(order); free(dS); free(pr); free(un); free(acc);
    return rc_all;
}
