/*
 * gfmc_oracle_dex.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain fp64 CPU oracle for the J_H -> infinity double-exchange Hamiltonian of
 * Eq. (2)-(3) -- the Hamiltonian the paper actually runs
 * -- and for the bond form of the GFMC update,
 * Eq. (15)-(22).  SURVEY.md section 8(f) row f1.
 * Same rules as gfmc_oracle.c: written from the paper, step by step, no moment
 * doubling, no batching, no code shared with the CUDA path; only tests/,
 * __graft_entry__.smoke() and bench.py's CPU legs may use it.
 *
 * Conventions: site i = x + L*(y + L*z); H has dimension N = L^3 (one orbital per
 * site: the electron spin is locked to the classical spin); the 2x2 objects are in
 * the (non-orthonormal) pair of states {|o>, |v>} of Eq. (21), index 0 = o, 1 = v.
 * An overall energy scale t multiplies Eq. (2) (the paper has t = 1).
 *
 * Pins (tests/test_oracle_dex.py): Eq. (3) against the spinor overlap
 * <chi_i|chi_j> (|t_ij|^2 = (1 + S_i.S_j)/2), apply_H against an independently
 * built dense matrix, moments against dense eigh, the ferromagnetic band, gauge
 * invariance, Eq. (22) against the 7x7 determinant of Eq. (17) and against the
 * eigenvalue product of Eq. (12) with the exact resolvent, the unwrapped phase,
 * the exact Delta S_eff of Eq. (7) (loosely, large M), and a hand-rolled
 * Algorithm-1 loop for the sweep.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define ORACLE_PI 3.14159265358979323846264338327950288

/* from gfmc_oracle.c (same shared object): kernel damping + the series of Eq. (24)/(29) */
int gfmc_oracle_green(int M, int K, const cplx *mu, int kernel, double lambda,
                      double a, double b, double *E, cplx *Gt);
double gfmc_oracle_magnetization(int N, const double *S);

/* ---------------------------------------------------------------- bound
 * |t_ij| = cos(Theta_ij / 2) <= 1 (Theta_ij the angle between S_i and S_j), so every
 * Gershgorin disc of Eq. (2) has centre 0 and radius <= 6|t|: a = 6|t|, b = 0,
 * independent of the spins (same reading as the Eq. (1) path: the paper gives no
 * rescaling).                                                  */
void gfmc_oracle_dex_bounds(double t, double *a, double *b)
{
    *a = 6.0 * fabs(t);
    *b = 0.0;
}

/* ---------------------------------------------------------------- Eq. (3)
 * t_ij = cos((th_i - th_j)/2) cos((ph_i - ph_j)/2) + i cos((th_i + th_j)/2) sin((ph_i - ph_j)/2),
 * PAPER.md:55; th = polar angle = acos(S^z), ph = azimuth = atan2(S^y, S^x) in (-pi, pi].
 * out[0] = Re, out[1] = Im.                                                        */
void gfmc_oracle_dex_hopping(const double *Si, const double *Sj, double *out)
{
    double thi = acos(fmax(-1.0, fmin(1.0, Si[2]))), thj = acos(fmax(-1.0, fmin(1.0, Sj[2])));
    double phi = atan2(Si[1], Si[0]), phj = atan2(Sj[1], Sj[0]);
    out[0] = cos(0.5 * (thi - thj)) * cos(0.5 * (phi - phj));
    out[1] = cos(0.5 * (thi + thj)) * sin(0.5 * (phi - phj));
}

static cplx hop(const double *Si, const double *Sj)
{
    double o[2];
    gfmc_oracle_dex_hopping(Si, Sj, o);
    return o[0] + I * o[1];
}

static void neighbours(int L, int i, int nb[6])
{
    int xx = i % L, yy = (i / L) % L, z = i / (L * L);
    nb[0] = ((xx + 1) % L)     + L * (yy + L * z);
    nb[1] = ((xx + L - 1) % L) + L * (yy + L * z);
    nb[2] = xx + L * (((yy + 1) % L)     + L * z);
    nb[3] = xx + L * (((yy + L - 1) % L) + L * z);
    nb[4] = xx + L * (yy + L * ((z + 1) % L));
    nb[5] = xx + L * (yy + L * ((z + L - 1) % L));
}

/* ---------------------------------------------------------------- operator
 * Eq. (2):  H = -sum_<ij> t_ij (c+_i c_j + H.c.), so
 * <i|H|j> = -t * t_ij for nearest neighbours (t_ji = conj t_ij), periodic lattice,
 * all six directions summed (use L >= 3).                                          */
void gfmc_oracle_dex_apply_H(int L, double t, const double *S, const cplx *x, cplx *y)
{
    int N = L * L * L;
    for (int i = 0; i < N; ++i) {
        int nb[6];
        neighbours(L, i, nb);
        cplx acc = 0.0;
        for (int d = 0; d < 6; ++d) acc += hop(S + 3 * i, S + 3 * nb[d]) * x[nb[d]];
        y[i] = -t * acc;
    }
}

/* ---------------------------------------------------------------- Eq. (15), (21)
 * Delta = H' - H for S_o -> S'_o has the non-zero elements Delta_jo = <j|Delta|o>
 * = -t (t'_jo - t_jo) and Delta_oj = conj Delta_jo, j over the 6 neighbours of o.
 * |v> = Delta|o> = sum_j Delta_jo |j>.  nb[6] receives the neighbour sites,
 * v[6] the amplitudes Delta_jo (same direction order as neighbours()).             */
void gfmc_oracle_dex_v(int L, double t, const double *S, int site, const double *S_new,
                       int32_t *nb_out, cplx *v)
{
    int nb[6];
    neighbours(L, site, nb);
    for (int d = 0; d < 6; ++d) {
        cplx told = hop(S + 3 * nb[d], S + 3 * site);
        cplx tnew = hop(S + 3 * nb[d], S_new);
        v[d] = -t * (tnew - told);
        nb_out[d] = nb[d];
    }
}

/* ---------------------------------------------------------------- moments
 * Eq. (25)-(26), from the two start vectors |o> and |v> of
 * Eq. (21)-(22):  mu_m(alpha,beta) = <alpha|T_m(H~)|beta>, alpha, beta in {o, v};
 * <o|r> = r[o], <v|r> = sum_j conj(Delta_jo) r[j].  mu is [M][2][2].  M-1
 * applications of H per start vector, direct read-out (no doubling).  |v> is NOT
 * normalised (mu_0(v,v) = <v|v>).                                                  */
int gfmc_oracle_dex_moments(int L, double t, const double *S, int site, const double *S_new,
                            int M, cplx *mu)
{
    int N = L * L * L;
    double a, b;
    gfmc_oracle_dex_bounds(t, &a, &b);
    if (site < 0 || site >= N || M < 1 || L < 3) return -1;
    int32_t nb[6];
    cplx v[6];
    gfmc_oracle_dex_v(L, t, S, site, S_new, nb, v);
    cplx *r0 = malloc(sizeof(cplx) * N), *r1 = malloc(sizeof(cplx) * N), *hx = malloc(sizeof(cplx) * N);
    if (!r0 || !r1 || !hx) { free(r0); free(r1); free(hx); return -2; }
    for (int beta = 0; beta < 2; ++beta) {
        memset(r0, 0, sizeof(cplx) * N);
        if (beta == 0) r0[site] = 1.0;
        else for (int d = 0; d < 6; ++d) r0[nb[d]] += v[d];
        for (int m = 0; m < M; ++m) {
            const cplx *r;
            if (m == 0) r = r0;
            else if (m == 1) {
                gfmc_oracle_dex_apply_H(L, t, S, r0, hx);
                for (int j = 0; j < N; ++j) r1[j] = (hx[j] - b * r0[j]) / a;
                r = r1;
            } else {
                gfmc_oracle_dex_apply_H(L, t, S, r1, hx);
                for (int j = 0; j < N; ++j) {
                    cplx nxt = 2.0 * ((hx[j] - b * r1[j]) / a) - r0[j];      /* Eq. (26) */
                    r0[j] = r1[j];
                    r1[j] = nxt;
                }
                r = r1;
            }
            cplx ov = 0.0;
            for (int d = 0; d < 6; ++d) ov += conj(v[d]) * r[nb[d]];
            mu[(m * 2 + 0) * 2 + beta] = r[site];
            mu[(m * 2 + 1) * 2 + beta] = ov;
        }
    }
    free(r0); free(r1); free(hx);
    return 0;
}

int gfmc_oracle_dex_moments_many(int L, double t, const double *S, const int32_t *sites, int n,
                                 const double *S_new /*[n][3]*/, int M, cplx *mu, int nthreads)
{
    int rc = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int s = 0; s < n; ++s) {
        int r = gfmc_oracle_dex_moments(L, t, S, sites[s], S_new + 3 * s, M, mu + (size_t)s * M * 4);
        if (r != 0) {
#ifdef _OPENMP
#pragma omp critical
#endif
            rc = r;
        }
    }
    return rc;
}

static double fermi(double E, double beta, double mu_chem)
{
    double x = beta * (E - mu_chem);
    if (x > 0.0) { double e = exp(-x); return e / (1.0 + e); }
    return 1.0 / (1.0 + exp(x));
}

/* ---------------------------------------------------------------- Eq. (22) + Eq. (14)
 * Gt is G~ [K][2][2] in {o, v} from gfmc_oracle_green (physical G = G~/a; v carries
 * physical units).  d_k = [1 + G_ov][1 + G_vo] - G_oo G_vv (Eq. (22)),
 * continuous phase from the top of the band and the Gauss-Chebyshev midpoint rule
 * exactly as in gfmc_oracle_delta_S (readings 10, 11).                              */
double gfmc_oracle_dex_delta_S(int K, const cplx *Gt, double a, double b, double T, double mu_chem,
                               double *theta_out, cplx *d_out)
{
    double beta = 1.0 / T;
    double sum = 0.0, theta = 0.0;
    cplx dprev = 1.0;
    for (int k = 0; k < K; ++k) {
        cplx Goo = Gt[4 * k + 0] / a, Gov = Gt[4 * k + 1] / a, Gvo = Gt[4 * k + 2] / a, Gvv = Gt[4 * k + 3] / a;
        cplx d = (1.0 + Gov) * (1.0 + Gvo) - Goo * Gvv;
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

int gfmc_oracle_dex_site_dS(int L, double t, double T, double mu_chem, int M, int K, int kernel,
                            double lambda, const double *S, int site, const double *S_new, double *dS)
{
    double a, b;
    gfmc_oracle_dex_bounds(t, &a, &b);
    cplx *mu = malloc(sizeof(cplx) * M * 4), *Gt = malloc(sizeof(cplx) * K * 4);
    if (!mu || !Gt) { free(mu); free(Gt); return -2; }
    int rc = gfmc_oracle_dex_moments(L, t, S, site, S_new, M, mu);
    if (rc == 0) rc = gfmc_oracle_green(M, K, mu, kernel, lambda, a, b, NULL, Gt);
    if (rc == 0) *dS = gfmc_oracle_dex_delta_S(K, Gt, a, b, T, mu_chem, NULL, NULL);
    free(mu); free(Gt);
    return rc;
}

/* ---------------------------------------------------------------- sweep
 * Algorithm 1 with the same frozen-batch two-colour schedule as
 * gfmc_oracle_sweep.  Sites of one colour are never nearest neighbours, so no bond
 * is touched by two flips of a batch and Delta of the joint flip is the sum of the
 * single-site Deltas; batch_sites = 1 is the paper's sequential algorithm.        */
int gfmc_oracle_dex_sweep(int L, double t, double T, double mu_chem, int M, int K, int kernel,
                          double lambda, double *S, int n_sweeps, int batch_sites,
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
                    int rc = gfmc_oracle_dex_site_dS(L, t, T, mu_chem, M, K, kernel, lambda, S, i, prop + 3 * i, &v);
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
