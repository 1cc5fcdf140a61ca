// post.cuh -- the small kernels around the fused Chebyshev step.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gfmc {

// ------------------------------------------------------------------ spins AoS <-> SoA
__global__ void spins_aos_to_soa(const double* __restrict__ S, double* Sx, double* Sy, double* Sz, int N)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) { Sx[i] = S[3 * i]; Sy[i] = S[3 * i + 1]; Sz[i] = S[3 * i + 2]; }
}
__global__ void spins_soa_to_aos(const double* __restrict__ Sx, const double* __restrict__ Sy,
                                 const double* __restrict__ Sz, double* S, int N)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) { S[3 * i] = Sx[i]; S[3 * i + 1] = Sy[i]; S[3 * i + 2] = Sz[i]; }
}

// ------------------------------------------------------------------ a2: start vectors
// |r_0> = |o_p vi> for the two start vectors of every pair ("PrepareVector"; Eq. (26) line 1).
// R0 has been zeroed; layout R[z][p][y][c][x], c = 2*vi + s; the unit entry of start vector vi sits at s = vi.
__global__ void init_start_vectors(double2* R0, const int32_t* __restrict__ sites, int P, int L)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    int o = sites[p];
    int x = o % L, y = (o / L) % L, z = o / (L * L);
    size_t row = (((size_t)z * P + p) * L + y) * 4;
    R0[(row + 0) * L + x] = make_double2(1.0, 0.0);     // vi = 0, s = up
    R0[(row + 3) * L + x] = make_double2(1.0, 0.0);     // vi = 1, s = down
}

// ------------------------------------------------------------------ moments from Gram sums
// Eq. (27)-(28), in their 2x2 (off-diagonal) form (reading 18):
//   mu_{2m}(a,b)   = 2 <r^a_m|r^b_m>     - delta_ab
//   mu_{2m-1}(a,b) = 2 <r^a_{m-1}|r^b_m> - mu_1(a,b),   mu_1(a,b) = <r^a_0|r^b_1>
// gram: [M/2 steps][P][ntiles][8] = (Yuu, Ydd, Re Yud, Im Yud, Xuu, Xdd, Re Xud, Im Xud), tiles summed in index order.
// mu: [P][M][2][2] double2.
__global__ void finalize_moments(const double* __restrict__ gram, double2* __restrict__ mu,
                                 int P, int M, int ntiles)
{
    const int half = M / 2;
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)P * (half + 1)) return;
    int p = (int)(idx / (half + 1));
    int m = (int)(idx % (half + 1));
    double2* out = mu + (size_t)p * M * 4;
    if (m == 0) {
        out[0] = make_double2(1, 0); out[1] = make_double2(0, 0);
        out[2] = make_double2(0, 0); out[3] = make_double2(1, 0);
        return;
    }
    double g[8], g1[8];
    const size_t step_stride = (size_t)P * ntiles * 8;
    const double* src = gram + (size_t)(m - 1) * step_stride + (size_t)p * ntiles * 8;
    const double* src1 = gram + (size_t)p * ntiles * 8;
#pragma unroll
    for (int k = 0; k < 8; ++k) { g[k] = 0.0; g1[k] = 0.0; }
    for (int t = 0; t < ntiles; ++t)
#pragma unroll
        for (int k = 0; k < 8; ++k) { g[k] += src[t * 8 + k]; g1[k] += src1[t * 8 + k]; }
    // odd moment 2m-1
    double2 o_uu, o_dd, o_ud;
    if (m == 1) {
        o_uu = make_double2(g[4], 0); o_dd = make_double2(g[5], 0); o_ud = make_double2(g[6], g[7]);
    } else {
        o_uu = make_double2(2 * g[4] - g1[4], 0); o_dd = make_double2(2 * g[5] - g1[5], 0);
        o_ud = make_double2(2 * g[6] - g1[6], 2 * g[7] - g1[7]);
    }
    double2* od = out + (size_t)(2 * m - 1) * 4;
    od[0] = o_uu; od[1] = o_ud; od[2] = make_double2(o_ud.x, -o_ud.y); od[3] = o_dd;
    if (2 * m < M) {
        double2* ev = out + (size_t)(2 * m) * 4;
        ev[0] = make_double2(2 * g[0] - 1, 0);
        ev[1] = make_double2(2 * g[2], 2 * g[3]);
        ev[2] = make_double2(2 * g[2], -2 * g[3]);
        ev[3] = make_double2(2 * g[1] - 1, 0);
    }
}

// ------------------------------------------------------------------ particle-hole shortcut (kModeHund1)
// On an even-L periodic lattice A = Gamma (i sigma_y) K (Gamma_i = (-1)^(x+y+z), K = complex conjugation) obeys
// A H A^-1 = -H for Eq. (1) (the hopping changes sign under Gamma, S.sigma under i sigma_y K), hence
//   r^dn_n = -Gamma_o (-1)^n A r^up_n,   (A psi)[i] = Gamma_i (conj psi_dn[i], -conj psi_up[i]),
// and every Gram block of Eq. (27)-(28) follows from the up-start vector alone:
//   Ydd = Yuu, Yud = 0, Xdd = -Xuu, Xud(m) = s_m conj W_m,  s_m = -Gamma_o (-1)^m,  W_m = sum_i Gamma_i (u'_i d_i - d'_i u_i).
// Start vectors: slot = p / 2, q = p % 2, chunk 2q + s; only |o_p up> is stored.
__global__ void init_start_vectors_ph(double2* R0, const int32_t* __restrict__ sites, int P, int Pslots, int L)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    int o = sites[p];
    int x = o % L, y = (o / L) % L, z = o / (L * L);
    size_t row = (((size_t)z * Pslots + (p >> 1)) * L + y) * 4;
    R0[(row + 2 * (p & 1)) * L + x] = make_double2(1.0, 0.0);
}

// gram: [M/2 steps][Pslots][ntiles][8] = per q: (Y, X, Re W, Im W).  mu: [P][M][2][2].
__global__ void finalize_moments_ph(const double* __restrict__ gram, double2* __restrict__ mu, const int32_t* __restrict__ sites,
                                    int P, int Pslots, int M, int ntiles, int L)
{
    const int half = M / 2;
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)P * (half + 1)) return;
    int p = (int)(idx / (half + 1));
    int m = (int)(idx % (half + 1));
    double2* out = mu + (size_t)p * M * 4;
    if (m == 0) {
        out[0] = make_double2(1, 0); out[1] = make_double2(0, 0);
        out[2] = make_double2(0, 0); out[3] = make_double2(1, 0);
        return;
    }
    const int o = sites[p];
    const double gam_o = (((o % L) + ((o / L) % L) + (o / (L * L))) & 1) ? -1.0 : 1.0;
    const size_t step_stride = (size_t)Pslots * ntiles * 8;
    const double* src = gram + (size_t)(m - 1) * step_stride + (size_t)(p >> 1) * ntiles * 8 + 4 * (p & 1);
    const double* src1 = gram + (size_t)(p >> 1) * ntiles * 8 + 4 * (p & 1);
    double g[4] = {0, 0, 0, 0}, g1[4] = {0, 0, 0, 0};
    for (int t = 0; t < ntiles; ++t)
#pragma unroll
        for (int k = 0; k < 4; ++k) { g[k] += src[t * 8 + k]; g1[k] += src1[t * 8 + k]; }
    const double sm = (m & 1) ? gam_o : -gam_o;          // s_m = -Gamma_o (-1)^m
    const double s1 = gam_o;                             // s_1
    // X_ud(m) = s_m conj(W_m)
    const double2 xud = make_double2(sm * g[2], -sm * g[3]);
    const double2 xud1 = make_double2(s1 * g1[2], -s1 * g1[3]);
    double o_uu; double2 o_ud;
    if (m == 1) { o_uu = g[1]; o_ud = xud; }
    else { o_uu = 2 * g[1] - g1[1]; o_ud = make_double2(2 * xud.x - xud1.x, 2 * xud.y - xud1.y); }
    double2* od = out + (size_t)(2 * m - 1) * 4;
    od[0] = make_double2(o_uu, 0); od[1] = o_ud; od[2] = make_double2(o_ud.x, -o_ud.y); od[3] = make_double2(-o_uu, 0);
    if (2 * m < M) {
        double2* ev = out + (size_t)(2 * m) * 4;
        ev[0] = make_double2(2 * g[0] - 1, 0); ev[1] = make_double2(0, 0);
        ev[2] = make_double2(0, 0);            ev[3] = make_double2(2 * g[0] - 1, 0);
    }
}

// ------------------------------------------------------------------ J_H -> infinity (kModeDex): Eq. (2)-(3), (15)-(22)
// Spinor of the classical spin in the gauge that reproduces Eq. (3) as t_ij = chi_i^dagger chi_j:
//   chi = (cos(th/2) e^{-i ph/2}, sin(th/2) e^{+i ph/2}),  th = polar angle, ph = atan2(S^y, S^x).
// Half-angle functions from S directly (well conditioned at both poles): rho = |(S^x,S^y)|,
//   S^z >= 0: c = sqrt((1+S^z)/2), s = rho/(2c);   S^z < 0: s = sqrt((1-S^z)/2), c = rho/(2s).
__device__ __forceinline__ void spinor_of(double Sx, double Sy, double Sz, double2& cu, double2& cd)
{
    const double rho = sqrt(Sx * Sx + Sy * Sy);
    double c, s;
    if (Sz >= 0.0) { c = sqrt(0.5 * (1.0 + Sz)); s = rho / (2.0 * c); }
    else           { s = sqrt(0.5 * (1.0 - Sz)); c = rho / (2.0 * s); }
    double sh, ch;
    sincos(0.5 * atan2(Sy, Sx), &sh, &ch);
    cu = make_double2(c * ch, -c * sh);
    cd = make_double2(s * ch, s * sh);
}
// chi_a^dagger chi_b
__device__ __forceinline__ double2 spinor_overlap(double2 au, double2 ad, double2 bu, double2 bd)
{
    return make_double2(au.x * bu.x + au.y * bu.y + ad.x * bd.x + ad.y * bd.y,
                        au.x * bu.y - au.y * bu.x + ad.x * bd.y - ad.y * bd.x);
}

// forward bond amplitudes T_d[i] = t_{i, i+e_d} for every site (recomputed after every accepted batch: N sites, negligible);
// written twice: direction-major Tx/Ty/Tz [N] (gfmc_hopping, resident kernel, run-time-L streaming kernel) and interleaved per
// lattice row Tq[z][y][d][x], d = (z-, x-, y-bond) (per-warp bond rings of the streaming kernel, cheb_step.cuh)
__global__ void dex_bonds_kernel(const double* __restrict__ Sx, const double* __restrict__ Sy, const double* __restrict__ Sz,
                                 double2* Tx, double2* Ty, double2* Tz, double2* Tq, int L)
{
    const int N = L * L * L;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int x = i % L, y = (i / L) % L, z = i / (L * L);
    const int jx = (x + 1) % L + L * (y + L * z), jy = x + L * ((y + 1) % L + L * z), jz = x + L * (y + L * ((z + 1) % L));
    double2 cu, cd, bu, bd;
    spinor_of(Sx[i], Sy[i], Sz[i], cu, cd);
    double2* row = Tq + (size_t)(i / L) * 3 * L + x;
    double2 tb;
    spinor_of(Sx[jx], Sy[jx], Sz[jx], bu, bd); tb = spinor_overlap(cu, cd, bu, bd); Tx[i] = tb; row[L] = tb;
    spinor_of(Sx[jy], Sy[jy], Sz[jy], bu, bd); tb = spinor_overlap(cu, cd, bu, bd); Ty[i] = tb; row[2 * L] = tb;
    spinor_of(Sx[jz], Sy[jz], Sz[jz], bu, bd); tb = spinor_overlap(cu, cd, bu, bd); Tz[i] = tb; row[0] = tb;
}

// Start vectors of Eq. (21)-(22): |o_p> in chunk 2q, |v_p> = Delta|o_p> = sum_j Delta_jo |j> in chunk 2q+1 (slot = p/2, q = p%2),
// Delta_jo = -t (t'_jo - t_jo) = -t chi_j^dagger (chi'_o - chi_o) over the six neighbours j of o (Eq. (15)).
// R0 has been zeroed.  Contributions to the same neighbour (L = 2 only) are added in direction order by the one thread.
// vnorm2[p] = <v|v> (mu_0(v,v)).
__global__ void init_start_vectors_dex(double2* R0, const int32_t* __restrict__ sites, const double* __restrict__ proposals, int by_site,
                                       const double* __restrict__ Sx, const double* __restrict__ Sy, const double* __restrict__ Sz,
                                       double t, double* vnorm2, int P, int Pslots, int L)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    const int o = sites[p];
    const int x = o % L, y = (o / L) % L, z = o / (L * L);
    const int slot = p >> 1, q = p & 1;
    auto at = [&](int xx, int yy, int zz, int c) -> double2& {
        return R0[((((size_t)zz * Pslots + slot) * L + yy) * 4 + c) * L + xx];
    };
    at(x, y, z, 2 * q) = make_double2(1.0, 0.0);
    const double* pr = proposals + 3 * (size_t)(by_site ? o : p);
    double2 ou, od, nu, nd;
    spinor_of(Sx[o], Sy[o], Sz[o], ou, od);
    spinor_of(pr[0], pr[1], pr[2], nu, nd);
    const double2 du = make_double2(nu.x - ou.x, nu.y - ou.y), dd = make_double2(nd.x - od.x, nd.y - od.y);
    const int nx[6] = {(x + 1) % L, (x + L - 1) % L, x, x, x, x};
    const int ny[6] = {y, y, (y + 1) % L, (y + L - 1) % L, y, y};
    const int nz[6] = {z, z, z, z, (z + 1) % L, (z + L - 1) % L};
    double n2 = 0.0;
    for (int d = 0; d < 6; ++d) {
        const int j = nx[d] + L * (ny[d] + L * nz[d]);
        double2 ju, jd;
        spinor_of(Sx[j], Sy[j], Sz[j], ju, jd);
        const double2 ov = spinor_overlap(ju, jd, du, dd);
        const double2 v = make_double2(-t * ov.x, -t * ov.y);
        double2& dst = at(nx[d], ny[d], nz[d], 2 * q + 1);
        dst = make_double2(dst.x + v.x, dst.y + v.y);
        n2 += v.x * v.x + v.y * v.y;
    }
    vnorm2[p] = n2;
}

// gram: [M/2 steps][Pslots][ntiles][16] = per q: (Yoo, Yvv, Re Yov, Im Yov, Xoo, Xvv, Re Xov, Im Xov).  mu [P][M][2][2] in {o, v}:
//   mu_{2m}(a,b) = 2 Y_m(a,b) - mu_0(a,b),  mu_0 = [[1, 0], [0, <v|v>]];  mu_{2m-1}(a,b) = 2 X_m(a,b) - mu_1(a,b),  mu_1 = X_1.
__global__ void finalize_moments_dex(const double* __restrict__ gram, double2* __restrict__ mu, const double* __restrict__ vnorm2,
                                     int P, int Pslots, int M, int ntiles)
{
    const int half = M / 2;
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)P * (half + 1)) return;
    int p = (int)(idx / (half + 1));
    int m = (int)(idx % (half + 1));
    double2* out = mu + (size_t)p * M * 4;
    const double vv = vnorm2[p];
    if (m == 0) {
        out[0] = make_double2(1, 0); out[1] = make_double2(0, 0);
        out[2] = make_double2(0, 0); out[3] = make_double2(vv, 0);
        return;
    }
    double g[8], g1[8];
    const size_t step_stride = (size_t)Pslots * ntiles * 16;
    const double* src = gram + (size_t)(m - 1) * step_stride + (size_t)(p >> 1) * ntiles * 16 + 8 * (p & 1);
    const double* src1 = gram + (size_t)(p >> 1) * ntiles * 16 + 8 * (p & 1);
#pragma unroll
    for (int k = 0; k < 8; ++k) { g[k] = 0.0; g1[k] = 0.0; }
    for (int t = 0; t < ntiles; ++t)
#pragma unroll
        for (int k = 0; k < 8; ++k) { g[k] += src[t * 16 + k]; g1[k] += src1[t * 16 + k]; }
    double2 o_oo, o_vv, o_ov;
    if (m == 1) {
        o_oo = make_double2(g[4], 0); o_vv = make_double2(g[5], 0); o_ov = make_double2(g[6], g[7]);
    } else {
        o_oo = make_double2(2 * g[4] - g1[4], 0); o_vv = make_double2(2 * g[5] - g1[5], 0);
        o_ov = make_double2(2 * g[6] - g1[6], 2 * g[7] - g1[7]);
    }
    double2* od = out + (size_t)(2 * m - 1) * 4;
    od[0] = o_oo; od[1] = o_ov; od[2] = make_double2(o_ov.x, -o_ov.y); od[3] = o_vv;
    if (2 * m < M) {
        double2* ev = out + (size_t)(2 * m) * 4;
        ev[0] = make_double2(2 * g[0] - 1, 0);
        ev[1] = make_double2(2 * g[2], 2 * g[3]);
        ev[2] = make_double2(2 * g[2], -2 * g[3]);
        ev[3] = make_double2(2 * g[1] - vv, 0);
    }
}

// ------------------------------------------------------------------ a4-a6: damping, G~ on the grid, Delta S_eff
struct GreenArgs {
    const double2* mu;        // [n][M][4] undamped moments
    const double*  w;         // [M] damping weights: w_0 = g_0/2, w_m = g_m  (Eq. (30))
    const double2* tw;        // [4K] twiddles exp(-i pi p/(2K))
    double2*       G;         // optional output [n][K][4], physical units (G~/a); may be null
    const int32_t* sites;     // [n]
    const double*  Sx; const double* Sy; const double* Sz;
    const double*  proposals; // [.][3]; null -> only G is produced
    double*        dS;        // [n] (indexed by j) output
    int by_site;              // proposals indexed by site (sweep) or by j
    int dex;                  // 1: the 2x2 block is in {o, v} and d is Eq. (22): Delta~ = sigma_x / a
    int n, M, K, Mc;
    double a, b, JH, beta, mu_chem;
};

constexpr int kGreenThreads = 256;

__device__ __forceinline__ double fermi_fn(double E, double beta, double mu_chem)
{
    double x = beta * (E - mu_chem);
    if (x > 0.0) { double e = exp(-x); return e / (1.0 + e); }
    return 1.0 / (1.0 + exp(x));
}

// Delta~ of the trial move in the 2x2 block of the updated site (on-site form of Eq. (17)-(22))
struct GreenDelta { double2 D00, D01, D10, D11; };
__device__ __forceinline__ void green_delta(const GreenArgs& a, int j, bool want_dS, GreenDelta& D)
{
    D.D00 = D.D01 = D.D10 = D.D11 = make_double2(0.0, 0.0);
    if (want_dS && a.dex) {
        // Eq. (22): d = (1 + G_ov)(1 + G_vo) - G_oo G_vv = det(1_2 + G [[0,1],[1,0]]),  G = G~/a
        D.D01 = make_double2(1.0 / a.a, 0.0); D.D10 = make_double2(1.0 / a.a, 0.0);
    } else if (want_dS) {
        const int site = a.sites[j];
        const double* pr = a.proposals + 3 * (size_t)(a.by_site ? site : j);
        const double c = a.JH / a.a;
        const double dx = pr[0] - a.Sx[site], dy = pr[1] - a.Sy[site], dz = pr[2] - a.Sz[site];
        D.D00 = make_double2(c * dz, 0.0); D.D01 = make_double2(c * dx, -c * dy);
        D.D10 = make_double2(c * dx, c * dy); D.D11 = make_double2(-c * dz, 0.0);
    }
}

// energy point k of site j from the four sums acc[e] = sum_m mu'_m(e) exp(-i m phi_k): G~ = (2i / sin phi_k) acc (Eq. (24) line 2),
// optional output of G = G~/a, and d_k = det(1 + G~_k Delta~) (Eq. (11))
__device__ __forceinline__ void green_point(const GreenArgs& a, int j, int k, const double2 (&acc)[4], bool want_dS, const GreenDelta& D, double2* sd)
{
    const int K = a.K;
    double sphi, cphi;
    sincospi((k + 0.5) / K, &sphi, &cphi);
    const double pre = 2.0 / sphi;
    double2 Gt[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) Gt[e] = make_double2(-pre * acc[e].y, pre * acc[e].x);
    if (a.G) {
        const double ia = 1.0 / a.a;
        double2* Go = a.G + ((size_t)j * K + k) * 4;
#pragma unroll
        for (int e = 0; e < 4; ++e) Go[e] = make_double2(Gt[e].x * ia, Gt[e].y * ia);
    }
    if (want_dS) {
        // A = G~ Delta~ ; d = (1 + A00)(1 + A11) - A01 A10
        auto cmul = [](double2 u, double2 v) { return make_double2(u.x * v.x - u.y * v.y, u.x * v.y + u.y * v.x); };
        auto cadd = [](double2 u, double2 v) { return make_double2(u.x + v.x, u.y + v.y); };
        double2 A00 = cadd(cmul(Gt[0], D.D00), cmul(Gt[1], D.D10));
        double2 A01 = cadd(cmul(Gt[0], D.D01), cmul(Gt[1], D.D11));
        double2 A10 = cadd(cmul(Gt[2], D.D00), cmul(Gt[3], D.D10));
        double2 A11 = cadd(cmul(Gt[2], D.D01), cmul(Gt[3], D.D11));
        A00.x += 1.0; A11.x += 1.0;
        double2 d1 = cmul(A00, A11), d2 = cmul(A01, A10);
        sd[k] = make_double2(d1.x - d2.x, d1.y - d2.y);
    }
}
__device__ __forceinline__ void green_finish(const GreenArgs& a, int j, const double2* sd, double* sth, double* sred);

// One CTA per site.  Direct O(M K) evaluation of the second line of Eq. (24) on the Chebyshev nodes
// (PAPER.md:162-164, 193, 197-201); then d_k = det(1 + G~_k Delta~) (Eq. (11); on-site 2x2 form),
// continuous phase from k = 0, and the Gauss-Chebyshev quadrature of Eq. (14).
__global__ void __launch_bounds__(kGreenThreads) green_dS_kernel(const GreenArgs a)
{
    extern __shared__ __align__(16) unsigned char gsm[];
    double2* smu = reinterpret_cast<double2*>(gsm);                      // [Mc][4]
    double2* sd = smu + (size_t)a.Mc * 4;                                // [K]
    double* sth = reinterpret_cast<double*>(sd + a.K);                   // [K]
    __shared__ double sred[kGreenThreads];

    const int j = blockIdx.x;
    const int tid = threadIdx.x;
    const int K = a.K, M = a.M;
    const double2* mu = a.mu + (size_t)j * M * 4;
    const bool want_dS = (a.proposals != nullptr);

    GreenDelta D;
    green_delta(a, j, want_dS, D);

    for (int kb = 0; kb < K; kb += kGreenThreads) {
        const int k = kb + tid;
        double2 acc[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[e] = make_double2(0.0, 0.0);
        const int fourK = 4 * K;
        const int stepk = (2 * k + 1) % fourK;
        int p = 0;
        for (int m0 = 0; m0 < M; m0 += a.Mc) {
            const int mc = min(a.Mc, M - m0);
            __syncthreads();
            for (int i = tid; i < mc * 4; i += kGreenThreads) {
                const double wm = a.w[m0 + (i >> 2)];
                const double2 v = mu[(size_t)m0 * 4 + i];
                smu[i] = make_double2(wm * v.x, wm * v.y);
            }
            __syncthreads();
            if (k < K) {
                for (int m = 0; m < mc; ++m) {
                    const double2 t = __ldg(a.tw + p);
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const double2 v = smu[m * 4 + e];
                        acc[e].x += v.x * t.x - v.y * t.y;
                        acc[e].y += v.x * t.y + v.y * t.x;
                    }
                    p += stepk; if (p >= fourK) p -= fourK;
                }
            }
        }
        if (k < K) green_point(a, j, k, acc, want_dS, D, sd);
    }
    if (!want_dS) return;
    __syncthreads();
    green_finish(a, j, sd, sth, sred);
}

// continuous phase + quadrature for one site; sd[K] holds d_k (all threads of the CTA call this after a __syncthreads)
__device__ __forceinline__ void green_finish(const GreenArgs& a, int j, const double2* sd, double* sth, double* sred)
{
    const int tid = threadIdx.x, K = a.K;
    // continuous phase: theta_0 = Arg d_0, theta_k = theta_{k-1} + Arg(d_k conj d_{k-1})
    const int kpt = (K + kGreenThreads - 1) / kGreenThreads;
    const int k0 = tid * kpt, k1 = min(K, k0 + kpt);
    double run = 0.0;
    for (int k = k0; k < k1; ++k) {
        const double2 d = sd[k];
        double inc;
        if (k == 0) inc = atan2(d.y, d.x);
        else { const double2 q = sd[k - 1]; inc = atan2(d.y * q.x - d.x * q.y, d.x * q.x + d.y * q.y); }
        run += inc;
        sth[k] = run;
    }
    sred[tid] = run;
    __syncthreads();
    // exclusive scan of the per-thread totals (256 values) by thread 0..: simple two-level
    if (tid == 0) {
        double s = 0.0;
        for (int t = 0; t < kGreenThreads; ++t) { double v = sred[t]; sred[t] = s; s += v; }
    }
    __syncthreads();
    const double base = sred[tid];
    double part = 0.0;
    for (int k = k0; k < k1; ++k) {
        double sphi, cphi;
        sincospi((k + 0.5) / K, &sphi, &cphi);
        const double E = a.a * cphi + a.b;
        part += fermi_fn(E, a.beta, a.mu_chem) * (base + sth[k]) * sphi;
    }
    __syncthreads();
    sred[tid] = part;
    __syncthreads();
    for (int off = kGreenThreads / 2; off > 0; off >>= 1) {
        if (tid < off) sred[tid] += sred[tid + off];
        __syncthreads();
    }
    if (tid == 0) a.dS[j] = a.beta * a.a / K * sred[0];
}

// ------------------------------------------------------------------ a5 by FFT (Eq. (29)-(32))
// The sums of Eq. (24) on the Chebyshev nodes are a discrete Fourier transform ("PerformsFFT"):
//     S_e(k) = sum_m mu'_m(e) exp(-i pi m (2k+1) / 2K) = sum_{m < 2K} [mu'_m(e) exp(-i pi m / 2K)] exp(-2 pi i m k / 2K),  k = 0 .. K-1,
// i.e. the first half of a 2K-point DFT of the pre-twiddled, zero-padded (or folded, if M > 2K) moment sequence.  The paper's index
// map chi_{2j+1} = gamma*_{M-j-1} folds this into a length-M real-to-complex transform and holds for REAL moments only
// (reading 19); the 2x2 blocks here have complex off-diagonal moments, so each of the four sequences gets its own complex
// transform.  One CTA per site, radix-2 decimation-in-frequency in shared memory (natural order in, bit-reversed out; the output of
// node k is read at the bit-reversed index, no reordering pass), twiddles from the same exact-argument table as the direct sum:
// exp(-2 pi i e / 2K) = tw[2e].  O(K log K) instead of O(M K) per site; needs K = 2^n and 6 K complex numbers of shared memory.
// Shared memory: work[2K] | out[4][K]; d_k and the phase scratch alias out[0] / out[1] once the four sums of a node have been read.
__global__ void __launch_bounds__(kGreenThreads) green_fft_dS_kernel(const GreenArgs a)
{
    extern __shared__ __align__(16) unsigned char gsm[];
    const int K = a.K, M = a.M, Nf = 2 * K;
    double2* work = reinterpret_cast<double2*>(gsm);          // [2K]
    double2* out = work + Nf;                                 // [4][K]
    double2* sd = out;                                        // aliases out[0]
    double* sth = reinterpret_cast<double*>(out + K);         // aliases out[1]
    __shared__ double sred[kGreenThreads];

    const int j = blockIdx.x, tid = threadIdx.x;
    const double2* mu = a.mu + (size_t)j * M * 4;
    const bool want_dS = (a.proposals != nullptr);
    GreenDelta D;
    green_delta(a, j, want_dS, D);
    const int logN = 31 - __clz(Nf);

    for (int e = 0; e < 4; ++e) {
        // pre-twiddled, damped moments: b(m) = w_m mu_m(e) exp(-i pi m / 2K); m >= 2K folds back (exp(-2 pi i m k / 2K) is 2K-periodic)
        for (int i = tid; i < Nf; i += kGreenThreads) {
            double2 b = make_double2(0.0, 0.0);
            for (int m = i; m < M; m += Nf) {
                const double wm = a.w[m];
                const double2 v = mu[(size_t)m * 4 + e];
                const double2 t = __ldg(a.tw + (m % (2 * Nf)));
                const double vx = wm * v.x, vy = wm * v.y;
                b.x += vx * t.x - vy * t.y; b.y += vx * t.y + vy * t.x;
            }
            work[i] = b;
        }
        __syncthreads();
        for (int half = Nf >> 1; half >= 1; half >>= 1) {
            const int tstride = Nf / half;                     // tw index of W^(j) at this stage: 2 * j * (Nf / (2 half))
            for (int b = tid; b < (Nf >> 1); b += kGreenThreads) {
                const int jj = b & (half - 1);
                const int i0 = ((b - jj) << 1) + jj;
                const double2 u = work[i0], v = work[i0 + half];
                work[i0] = make_double2(u.x + v.x, u.y + v.y);
                const double dx = u.x - v.x, dy = u.y - v.y;
                const double2 t = __ldg(a.tw + jj * tstride);
                work[i0 + half] = make_double2(dx * t.x - dy * t.y, dx * t.y + dy * t.x);
            }
            __syncthreads();
        }
        for (int k = tid; k < K; k += kGreenThreads) out[(size_t)e * K + k] = work[__brev((unsigned)k) >> (32 - logN)];
        __syncthreads();
    }
    for (int k = tid; k < K; k += kGreenThreads) {
        double2 acc[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[e] = out[(size_t)e * K + k];
        green_point(a, j, k, acc, want_dS, D, sd);             // writes sd[k] = out[0][k] after all four reads of this k
    }
    if (!want_dS) return;
    __syncthreads();
    green_finish(a, j, sd, sth, sred);
}

// ------------------------------------------------------------------ batch cursor of a sweep (CUDA-graph friendly site gather)
// The sites of the next batch are order[*cursor .. *cursor + P); the cursor advances on the device so that the whole per-batch launch
// sequence has constant arguments and can be replayed as one CUDA graph (launch-bound regime: small lattices, small batches).
__global__ void __launch_bounds__(1024) next_batch_kernel(const int32_t* __restrict__ order, int* cursor, int32_t* __restrict__ sites, int P)
{
    const int base = *cursor;
    for (int j = threadIdx.x; j < P; j += blockDim.x) sites[j] = order[base + j];
    __syncthreads();
    if (threadIdx.x == 0) *cursor = base + P;
}

// ------------------------------------------------------------------ a7: Metropolis accept + spin update
// accept iff -Delta S > ln u  (Alg. 1 line 10-12; reading 15).  All sites of the batch were
// evaluated against the same configuration; accepted flips are applied here together ("UpdateStatus", PAPER.md:339;
// matrix-free, so there is no H to patch).
struct MetropolisArgs {
    const int32_t* sites; const double* dS; const double* proposals; const double* uniforms;
    double* Sx; double* Sy; double* Sz;
    uint8_t* accepted;          // [n] by j, may be null
    double* dS_log;             // [N] by site, may be null
    uint8_t* accept_log;        // [N] by site, may be null
    unsigned long long* n_accepted;
    int n, by_site;
    int apply;                  // 1: accepted flips are written to the spin field; 0: decisions only (gfmc_decide_batch: the flips of a
                                // batch sharded over several GPUs are applied by gfmc_apply_flips once every rank's decisions are known)
};
__global__ void metropolis_kernel(const MetropolisArgs a)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= a.n) return;
    const int site = a.sites[j];
    const size_t q = a.by_site ? (size_t)site : (size_t)j;
    const double v = a.dS[j];
    const bool acc = (-v > log(a.uniforms[q]));
    if (a.accepted) a.accepted[j] = acc ? 1 : 0;
    if (a.dS_log) a.dS_log[site] = v;
    if (a.accept_log) a.accept_log[site] = acc ? 1 : 0;
    if (acc) {
        if (a.apply) { a.Sx[site] = a.proposals[3 * q]; a.Sy[site] = a.proposals[3 * q + 1]; a.Sz[site] = a.proposals[3 * q + 2]; }
        atomicAdd(a.n_accepted, 1ULL);
    }
}

// S_site <- proposals[j] for every listed site with accepted[j] != 0 ("UpdateStatus"; Alg. 1 lines 11-12) -- the second
// half of metropolis_kernel, for decisions taken elsewhere (another GPU's share of the batch).
__global__ void apply_flips_kernel(const int32_t* __restrict__ sites, const double* __restrict__ proposals, const uint8_t* __restrict__ accepted,
                                   int n, double* Sx, double* Sy, double* Sz, unsigned long long* n_accepted)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n || !accepted[j]) return;
    const int site = sites[j];
    Sx[site] = proposals[3 * (size_t)j]; Sy[site] = proposals[3 * (size_t)j + 1]; Sz[site] = proposals[3 * (size_t)j + 2];
    atomicAdd(n_accepted, 1ULL);
}

// ------------------------------------------------------------------ random trial moves of the Algorithm-1 driver
// Algorithm 1 "changes the spin randomly" (line 4) and compares with rand() (line 10); the generator is
// not specified.  DESIGN.md reading f3-1: counter-based Philox4x32-10 (Salmon et al., SC'11), key = (seed lo, seed hi),
// counter = (site, sweep lo, stream, sweep hi); stream 0 -> (u1, u2), stream 1 -> u3; 53-bit uniforms; proposal uniform on the
// sphere by the recipe of DESIGN.md §3; acceptance uniform 1 - u3 in (0,1].  Indexed by (sweep, site): any schedule draws the same numbers.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ __forceinline__ double u01_from_words(uint32_t w_even, uint32_t w_odd)
{
    return (double)((((unsigned long long)w_even << 32) | w_odd) >> 11) * 0x1.0p-53;
}
__global__ void propose_kernel(unsigned long long seed, unsigned long long sweep, int N, double* __restrict__ proposals, double* __restrict__ uniforms)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32), s0 = (uint32_t)sweep, s1 = (uint32_t)(sweep >> 32);
    uint32_t a[4], b[4];
    philox4x32_10((uint32_t)i, s0, 0u, s1, k0, k1, a);
    philox4x32_10((uint32_t)i, s0, 1u, s1, k0, k1, b);
    const double u1 = u01_from_words(a[0], a[1]), u2 = u01_from_words(a[2], a[3]), u3 = u01_from_words(b[0], b[1]);
    const double z = 2.0 * u1 - 1.0;
    const double r = sqrt(__dadd_rn(1.0, -__dmul_rn(z, z)));      // no FMA contraction: same roundings as the oracle's 1 - z*z
    double sn, cs;
    sincos(2.0 * 3.14159265358979323846 * u2, &sn, &cs);
    proposals[3 * (size_t)i] = r * cs; proposals[3 * (size_t)i + 1] = r * sn; proposals[3 * (size_t)i + 2] = z;
    uniforms[i] = 1.0 - u3;
}

// ------------------------------------------------------------------ a8: magnetization |sum_i S_i| / N
// (Alg. 1 line 15; "MeasureSpin").  One CTA, fixed summation order.
// run_stats (may be null): running statistics of the sweeps of one gfmc_run call, updated by thread 0 after the sweep's value is
// known -- Alg. 1 lines 16-17 ("M <- M + m", "return M/S") in Welford form: [0] = S (sweeps so far),
// [1] = mean of m, [2] = sum of squared deviations, [3] = accepted flips so far (from the sweep's counter *n_acc).
__global__ void __launch_bounds__(1024) magnetization_kernel(const double* __restrict__ Sx, const double* __restrict__ Sy,
                                                             const double* __restrict__ Sz, int N, double* out,
                                                             double* run_stats, const unsigned long long* n_acc)
{
    __shared__ double sx[1024], sy[1024], sz[1024];
    double ax = 0, ay = 0, az = 0;
    for (int i = threadIdx.x; i < N; i += 1024) { ax += Sx[i]; ay += Sy[i]; az += Sz[i]; }
    sx[threadIdx.x] = ax; sy[threadIdx.x] = ay; sz[threadIdx.x] = az;
    __syncthreads();
    for (int off = 512; off > 0; off >>= 1) {
        if (threadIdx.x < off) {
            sx[threadIdx.x] += sx[threadIdx.x + off]; sy[threadIdx.x] += sy[threadIdx.x + off]; sz[threadIdx.x] += sz[threadIdx.x + off];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double m = sqrt(sx[0] * sx[0] + sy[0] * sy[0] + sz[0] * sz[0]) / N;
        *out = m;
        if (run_stats) {
            const double n = run_stats[0] + 1.0, d = m - run_stats[1];
            const double mean = run_stats[1] + d / n;
            run_stats[0] = n; run_stats[1] = mean; run_stats[2] += d * (m - mean);
            run_stats[3] += (double)*n_acc;
        }
    }
}

}  // namespace gfmc
