// exact_batch.cuh -- exactness inside a batch, Hamiltonian of Eq. (1).
//
// The frozen batch evaluates every site of a batch against the configuration at batch start.  Here the sites of a batch are
// decided one after the other and site B sees the earlier ACCEPTED flips of the same batch exactly, without a new Chebyshev
// recursion: Eq. (11) for the pair (H + Delta_U, H + Delta_U + Delta_B), U = accepted sites so far, is
//     d_B|U(z) = det_2(1_2 + G_U,BB(z) Delta_B)                                  (the block reduction of Eq. (17)-(22))
// and the resolvent identity G_U = G - G Delta_U G_U gives the Green blocks of H + Delta_U between the sites of the batch from
// those at batch start.  The kernels below apply it one accepted site at a time (a rank-2 Woodbury update of every later block):
//     G_XY <- G_XY - G_XA W_A G_AY,   W_A = Delta_A (1_2 + G_AA Delta_A)^-1,   for all X, Y after A in the batch,
// so that when site B's turn comes G_BB already IS G_U,BB.  (The CPU checker used by the tests solves the full
// 2|U| x 2|U| system per site and energy instead: same algebra, different arithmetic.)
//
// The blocks at batch start come from CROSS moments mu_m(X a, Y b) = <o_X a| T_m(H~) |o_Y b> = r_m^{Y b}[X a]  (Eq. (25)-(26),
// PAPER.md:168-183), read out of the work vectors after every fused step (the doubling of Eq. (27)-(28) would need Gram sums
// between different slots, i.e. a (2P)^2 dot-product matrix per step, so this mode runs the plain M-1 steps), and from the same
// reconstruction kernels as the diagonal blocks (Eq. (24) is linear in the moments).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "post.cuh"

namespace gfmc {

// xmu[X][Y][m][al][be] = r_m^{Y be}[site X, component al]: work-vector layout R[z][p][y][c][x], p = Y, c = 2*be + al.
__global__ void cross_readout_kernel(const double2* __restrict__ R, const int32_t* __restrict__ sites, int P, int L, int M, int m,
                                     double2* __restrict__ xmu)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= P * P * 4) return;
    const int e = idx & 3, Y = (idx >> 2) % P, X = (idx >> 2) / P;
    const int al = e >> 1, be = e & 1;
    const int o = sites[X];
    const int x = o % L, y = (o / L) % L, z = o / (L * L);
    xmu[(((size_t)X * P + Y) * M + m) * 4 + e] = R[((((size_t)z * P + Y) * L + y) * 4 + (2 * be + al)) * L + x];
}

struct ExactArgs {
    double2* G;               // [P][P][K][4] physical Green blocks (G~/a), updated in place as flips are accepted
    const int32_t* sites;     // [P]
    const double* proposals; const double* uniforms; int by_site;
    double* Sx; double* Sy; double* Sz;
    double* dS;               // [P]
    uint8_t* accepted;        // [P] by position; always written (the update kernel reads it)
    double* dS_log; uint8_t* accept_log;      // [N] by site, may be null
    unsigned long long* n_accepted;
    unsigned int* bad;        // sticky error word of the batch: bit 0 = a non-finite Delta S, bit 1 = a singular 1 + G_jj Delta_j at some node
    int P, K, j;
    double a, b, JH, beta, mu_chem;
};

__device__ __forceinline__ double2 xb_mul(double2 u, double2 v) { return make_double2(u.x * v.x - u.y * v.y, u.x * v.y + u.y * v.x); }
__device__ __forceinline__ double2 xb_add(double2 u, double2 v) { return make_double2(u.x + v.x, u.y + v.y); }
__device__ __forceinline__ double2 xb_sub(double2 u, double2 v) { return make_double2(u.x - v.x, u.y - v.y); }
// C = A B for 2x2 complex blocks stored (00, 01, 10, 11)
__device__ __forceinline__ void xb_mm(const double2 (&A)[4], const double2 (&B)[4], double2 (&C)[4])
{
    C[0] = xb_add(xb_mul(A[0], B[0]), xb_mul(A[1], B[2])); C[1] = xb_add(xb_mul(A[0], B[1]), xb_mul(A[1], B[3]));
    C[2] = xb_add(xb_mul(A[2], B[0]), xb_mul(A[3], B[2])); C[3] = xb_add(xb_mul(A[2], B[1]), xb_mul(A[3], B[3]));
}
// physical Delta_j = J_H (S'_j - S_j).sigma of the trial at position j (S_j: the site's CURRENT spin, which no other trial touches)
__device__ __forceinline__ void exact_delta(const ExactArgs& a, int j, double2 (&D)[4])
{
    const int site = a.sites[j];
    const double* pr = a.proposals + 3 * (size_t)(a.by_site ? site : j);
    const double dx = pr[0] - a.Sx[site], dy = pr[1] - a.Sy[site], dz = pr[2] - a.Sz[site];
    D[0] = make_double2(a.JH * dz, 0.0); D[1] = make_double2(a.JH * dx, -a.JH * dy);
    D[2] = make_double2(a.JH * dx, a.JH * dy); D[3] = make_double2(-a.JH * dz, 0.0);
}

// Decision of site j (one CTA): d_k = det(1 + G_jj(k) Delta_j) on the K nodes, continuous phase, quadrature of Eq. (14), accept iff
// -Delta S > ln u (Alg. 1 line 10).  The spin is NOT written here (exact_update_kernel still needs the old one).
__global__ void __launch_bounds__(kGreenThreads) exact_decide_kernel(const ExactArgs a)
{
    extern __shared__ __align__(16) unsigned char gsm[];
    double2* sd = reinterpret_cast<double2*>(gsm);                       // [K]
    double* sth = reinterpret_cast<double*>(sd + a.K);                   // [K]
    __shared__ double sred[kGreenThreads];
    const int j = a.j, tid = threadIdx.x, K = a.K;
    double2 D[4];
    exact_delta(a, j, D);
    const double2* Gjj = a.G + ((size_t)j * a.P + j) * K * 4;
    for (int k = tid; k < K; k += kGreenThreads) {
        double2 G[4], A[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) G[e] = Gjj[(size_t)k * 4 + e];
        xb_mm(G, D, A);
        A[0].x += 1.0; A[3].x += 1.0;
        sd[k] = xb_sub(xb_mul(A[0], A[3]), xb_mul(A[1], A[2]));
    }
    __syncthreads();
    // green_finish wants the rescaled convention Delta S = (beta a / K) sum ...: it only uses a.a, a.b, a.beta, a.mu_chem, a.K, a.dS
    GreenArgs ga{};
    ga.K = K; ga.a = a.a; ga.b = a.b; ga.beta = a.beta; ga.mu_chem = a.mu_chem; ga.dS = a.dS;
    green_finish(ga, j, sd, sth, sred);
    __syncthreads();
    if (tid == 0) {
        const int site = a.sites[j];
        const size_t q = a.by_site ? (size_t)site : (size_t)j;
        const double v = a.dS[j];
        if (!isfinite(v)) atomicOr(a.bad, 1u);          // -NaN > ln u is false: without the flag such a site would be rejected silently
        const bool acc = (-v > log(a.uniforms[q]));
        a.accepted[j] = acc ? 1 : 0;
        if (a.dS_log) a.dS_log[site] = v;
        if (a.accept_log) a.accept_log[site] = acc ? 1 : 0;
        if (acc) atomicAdd(a.n_accepted, 1ULL);
    }
}

// If site j was accepted: G_XY(k) -= G_Xj(k) W(k) G_jY(k) for every X, Y > j, W = Delta_j (1 + G_jj Delta_j)^-1.  The blocks in row j
// and column j are only read, so the update is race-free.  One thread per (X, Y, k).
__global__ void exact_update_kernel(const ExactArgs a)
{
    const int j = a.j, P = a.P, K = a.K;
    if (!a.accepted[j]) return;
    const int rest = P - j - 1;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)rest * rest * K) return;
    const int k = (int)(idx % K);
    const int xy = (int)(idx / K);
    const int X = j + 1 + xy / rest, Y = j + 1 + xy % rest;
    double2 D[4], Gjj[4], A[4], W[4], GXj[4], GjY[4], T1[4], T2[4];
    exact_delta(a, j, D);
    const double2* base = a.G;
    auto blk = [&](int r, int c) { return base + (((size_t)r * P + c) * K + k) * 4; };
#pragma unroll
    for (int e = 0; e < 4; ++e) { Gjj[e] = blk(j, j)[e]; GXj[e] = blk(X, j)[e]; GjY[e] = blk(j, Y)[e]; }
    xb_mm(Gjj, D, A);
    A[0].x += 1.0; A[3].x += 1.0;
    // inverse of the 2x2 block A
    const double2 det = xb_sub(xb_mul(A[0], A[3]), xb_mul(A[1], A[2]));
    const double dn = det.x * det.x + det.y * det.y;
    if (!(dn > 0.0) || !isfinite(dn)) { atomicOr(a.bad, 2u); return; }      // d_k = 0 (or NaN) at this node: no inverse; the host reports it
    const double2 idet = make_double2(det.x / dn, -det.y / dn);
    double2 Ai[4];
    Ai[0] = xb_mul(A[3], idet); Ai[3] = xb_mul(A[0], idet);
    Ai[1] = xb_mul(make_double2(-A[1].x, -A[1].y), idet); Ai[2] = xb_mul(make_double2(-A[2].x, -A[2].y), idet);
    xb_mm(D, Ai, W);
    xb_mm(GXj, W, T1);
    xb_mm(T1, GjY, T2);
    double2* out = a.G + (((size_t)X * P + Y) * K + k) * 4;
#pragma unroll
    for (int e = 0; e < 4; ++e) out[e] = xb_sub(out[e], T2[e]);
}

// After the last decision: write the accepted trial spins (all together, like the frozen batch's metropolis_kernel).
__global__ void exact_apply_kernel(const ExactArgs a)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= a.P || !a.accepted[j]) return;
    const int site = a.sites[j];
    const size_t q = a.by_site ? (size_t)site : (size_t)j;
    a.Sx[site] = a.proposals[3 * q]; a.Sy[site] = a.proposals[3 * q + 1]; a.Sz[site] = a.proposals[3 * q + 2];
}

}  // namespace gfmc
