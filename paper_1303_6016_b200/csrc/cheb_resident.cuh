// cheb_resident.cuh -- the fused Chebyshev recursion for SMALL lattices (L <= 12), vectors resident in shared memory.
//
// Same arithmetic as cheb_step.cuh: Eq. (26) with H of Eq. (1) -- or of
// Eq. (2)-(3) (kModeDex: complex bond amplitudes, start vectors |o>, |v> of Eq. (21)) -- applied matrix-free, and
// the Gram blocks of Eq. (27)-(28) per step.  What differs is where the vectors live.  For L <= 12 both work
// vectors of a slot (r_{m-1}, r_{m-2}: 2 x 4 chunks x N complex fp64 = 128 N bytes: 64 KiB at L = 8, 216 KiB at L = 12) fit in
// the shared memory of ONE CTA, so the whole recursion m = 1 .. M/2 runs inside one launch with NO global-memory traffic for the
// vectors: start vectors are written in shared memory (row a2), every step reads its 6 neighbours + own site from the resident
// r_{m-1}, overwrites the resident r_{m-2} in place, and only the Gram sums per slot and step leave the SM.  One __syncthreads per
// step.  This is the "vectors resident on chip" design of SURVEY.md §8(f2) for the lattices where it fits one SM; the streaming
// kernel of cheb_step.cuh is launch/latency-bound there (config 2: 29 us per step for 25 MB of algorithmic traffic).
//
// Layout in shared memory: buf[b][g][c][i] (double2), b = ping-pong buffer, g = slot inside the CTA (G = 512 / roundup(N, 32)
// slots per CTA), c = chunk (kModeHund2: 2*vi + s; kModeHund1: 2*q + s; kModeDex: 2*q + vi, see cheb_step.cuh), i = site
// x + L (y + L z).  A warp reads 32 consecutive double2 = 512 contiguous bytes: conflict-free.  Thread (g, i) owns site i of slot g
// for the whole recursion; its spin and its 6 neighbour indices stay in registers.  For 512 < N <= 1728 (L = 9 .. 12) a CTA holds
// one slot and a thread owns up to four sites (template parameter SPT).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "cheb_step.cuh"

namespace gfmc {

constexpr int kResThreads = 512;
constexpr int kResWarps = kResThreads / 32;

struct ResidentArgs {
    const int32_t* sites;    // [P] start sites (device)
    const double*  Sx;       // spin field, SoA [N]
    const double*  Sy;
    const double*  Sz;
    const double2* Tx;       // kModeDex: forward bond amplitudes t_{i,i+e_d} of Eq. (3), SoA [N] per direction
    const double2* Ty;
    const double2* Tz;
    const double2* R0;       // kModeDex: start vectors |o_q>, |v_q> as written by init_start_vectors_dex (layout R[z][p][y][c][x])
    double*        gram;     // [nsteps][Ps][NG] partial Gram sums (one tile per slot), NG = gram_width(MODE)
    double t_over_a;         // t / a
    double jh_over_a;        // J_H / a
    int L, N, Npad;          // lattice edge, sites, sites rounded up to a multiple of 32
    int G;                   // slots per CTA
    int P, Ps;               // start sites, slots (kModeHund2: Ps = P; kModeHund1: Ps = ceil(P / 2))
    int nsteps;              // M / 2
};

__host__ __device__ inline size_t resident_smem_bytes(int N, int G)
{
    return (size_t)2 * G * 4 * N * sizeof(double2) + (size_t)2 * kResWarps * 16 * sizeof(double);
}

// sum of 8 values over the 32 lanes of a warp with 9 double shuffles: each level halves the number of values a lane carries.
// On return lane l holds the warp total of value index (l >> 2).  Fixed order: bit-reproducible.
__device__ __forceinline__ double warp_reduce8(const double (&v)[8], int lane)
{
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
    double w[4], u[2];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const double send = b4 ? v[j] : v[j + 4], keep = b4 ? v[j + 4] : v[j];
        w[j] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const double send = b3 ? w[j] : w[j + 2], keep = b3 ? w[j + 2] : w[j];
        u[j] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    const double send = b2 ? u[0] : u[1], keep = b2 ? u[1] : u[0];
    double s = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    return s;
}

// SPT = sites per thread.  SPT == 1 (N <= 512): G slots per CTA, thread (g, i) owns site i of slot g.  SPT > 1 (512 < N <= 1728,
// i.e. L = 9 .. 12, one slot per CTA): thread t owns sites t, t + 512, ...; its spins stay in registers, neighbour indices are packed
// two per register, and (kModeDex) the bond amplitudes are re-read from the L2-resident tables every step instead of living in registers.
template <int MODE, int SPT>
__global__ void __launch_bounds__(kResThreads, 1) cheb_resident_kernel(const __grid_constant__ ResidentArgs a)
{
    constexpr int NG = gram_width(MODE);
    constexpr bool kBondsInRegs = (SPT == 1);
    extern __shared__ __align__(16) unsigned char res_smem[];
    double2* buf = reinterpret_cast<double2*>(res_smem);
    const int N = a.N, L = a.L, G = a.G;
    double* red = reinterpret_cast<double*>(buf + (size_t)2 * G * 4 * N);      // [2][kResWarps][16]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = (SPT == 1) ? tid / a.Npad : 0;
    const int slot = blockIdx.x * G + g;

    // a2: start vectors, written straight into the resident buffer 0 ("PrepareVector"; Eq. (26) line 1)
    for (int k = tid; k < 2 * G * 4 * N; k += kResThreads) buf[k] = make_double2(0.0, 0.0);
    __syncthreads();
    if (tid < G && blockIdx.x * G + tid < a.Ps) {
        const int s = blockIdx.x * G + tid;
        double2* b0 = buf + (size_t)tid * 4 * N;
        if (MODE == kModeHund2) {
            const int o = a.sites[s];
            b0[0 * N + o] = make_double2(1.0, 0.0);          // |o up>  : vi = 0, s = up
            b0[3 * N + o] = make_double2(1.0, 0.0);          // |o down>: vi = 1, s = down
        } else if (MODE == kModeHund1) {
#pragma unroll
            for (int q = 0; q < 2; ++q)
                if (2 * s + q < a.P) b0[(2 * q) * N + a.sites[2 * s + q]] = make_double2(1.0, 0.0);   // |o_q up>
        }
    }

    // this thread's sites: neighbours (packed two per register), spin, sublattice sign -- constant over the whole recursion
    int site[SPT], nbx[SPT], nby[SPT], nbz[SPT];
    bool act[SPT];
    double sx[SPT], sy[SPT], sz[SPT], gam[SPT];
    double2 txf, txb, tyf, tyb, tzf, tzb;                    // kModeDex with SPT == 1 only
#pragma unroll
    for (int j = 0; j < SPT; ++j) {
        const int i = (SPT == 1) ? tid - g * a.Npad : tid + j * kResThreads;
        act[j] = (g < G) && (i < N) && (slot < a.Ps);
        const int ii = act[j] ? i : 0;
        site[j] = ii;
        const int x = ii % L, y = (ii / L) % L, z = ii / (L * L);
        const int n_xm = ii - x + (x + L - 1) % L, n_xp = ii - x + (x + 1) % L;
        const int n_ym = ii + (((y + L - 1) % L) - y) * L, n_yp = ii + (((y + 1) % L) - y) * L;
        const int n_zm = ii + (((z + L - 1) % L) - z) * L * L, n_zp = ii + (((z + 1) % L) - z) * L * L;
        nbx[j] = n_xm | (n_xp << 16); nby[j] = n_ym | (n_yp << 16); nbz[j] = n_zm | (n_zp << 16);
        gam[j] = ((x + y + z) & 1) ? -1.0 : 1.0;
        sx[j] = sy[j] = sz[j] = 0.0;
        if (MODE != kModeDex) { sx[j] = a.Sx[ii]; sy[j] = a.Sy[ii]; sz[j] = a.Sz[ii]; }
        else {
            if (act[j]) {
                // |o_q>, |v_q> = Delta|o_q> (Eq. (21)) were written by init_start_vectors_dex in the streaming layout
                const double2* src = a.R0 + ((((size_t)z * a.Ps + slot) * L + y) * 4) * L + x;
                double2* b0 = buf + (size_t)g * 4 * N;
#pragma unroll
                for (int k = 0; k < 4; ++k) b0[k * N + ii] = src[k * L];
            }
            if (kBondsInRegs) {
                // bond amplitudes of this site (Eq. (3)): forward t_{i,i+e}; backward t_{i,i-e} = conj(forward bond of the neighbour)
                txf = a.Tx[ii]; txb = a.Tx[n_xm]; tyf = a.Ty[ii]; tyb = a.Ty[n_ym]; tzf = a.Tz[ii]; tzb = a.Tz[n_zm];
            }
        }
    }
    const int wps = (SPT == 1) ? a.Npad / 32 : kResWarps;     // warps per slot
    __syncthreads();

    for (int m = 1; m <= a.nsteps; ++m) {
        const double scale = (m == 1) ? 1.0 : 2.0;
        const double ct = -scale * a.t_over_a;
        const double cj = scale * a.jh_over_a;
        const double2* cur = buf + ((size_t)((m - 1) & 1) * G + g) * 4 * N;      // r_{m-1}
        double2* nxt = buf + ((size_t)(m & 1) * G + g) * 4 * N;                  // r_{m-2} on entry, r_m on exit
        double gs[NG];
#pragma unroll
        for (int k = 0; k < NG; ++k) gs[k] = 0.0;
#pragma unroll
        for (int j = 0; j < SPT; ++j) {
            if (!act[j]) continue;
            const int ii = site[j];
            const int n_xm = nbx[j] & 0xffff, n_xp = nbx[j] >> 16, n_ym = nby[j] & 0xffff, n_yp = nby[j] >> 16;
            const int n_zm = nbz[j] & 0xffff, n_zp = nbz[j] >> 16;
            if (MODE == kModeDex && !kBondsInRegs) {
                txf = __ldg(a.Tx + ii); txb = __ldg(a.Tx + n_xm); tyf = __ldg(a.Ty + ii); tyb = __ldg(a.Ty + n_ym);
                tzf = __ldg(a.Tz + ii); tzb = __ldg(a.Tz + n_zm);
            }
            double2 acc[4], c0[4], nx[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double2* ck = cur + k * N;
                if (MODE != kModeDex)
                    acc[k] = add2(add2(add2(ck[n_zm], ck[n_zp]), add2(ck[n_xm], ck[n_xp])), add2(ck[n_ym], ck[n_yp]));
                else    // sum_j t_ij x_j over the six bonds (Eq. (2)-(3)), same order as cheb_step.cuh
                    acc[k] = add2(add2(add2(cmulc(tzb, ck[n_zm]), cmul(tzf, ck[n_zp])), add2(cmulc(txb, ck[n_xm]), cmul(txf, ck[n_xp]))),
                                  add2(cmulc(tyb, ck[n_ym]), cmul(tyf, ck[n_yp])));
                c0[k] = ck[ii];
            }
            if (MODE == kModeDex) {
#pragma unroll
                for (int k = 0; k < 4; ++k) { nx[k].x = ct * acc[k].x; nx[k].y = ct * acc[k].y; }
            } else {
                const double hx = cj * sx[j], hy = cj * sy[j], hz = cj * sz[j];
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    const double2 u = c0[2 * v], d = c0[2 * v + 1];
                    // (h.sigma) (u,d)^T : up = hz u + (hx - i hy) d ; down = (hx + i hy) u - hz d
                    nx[2 * v].x = ct * acc[2 * v].x + (hz * u.x + hx * d.x + hy * d.y);
                    nx[2 * v].y = ct * acc[2 * v].y + (hz * u.y + hx * d.y - hy * d.x);
                    nx[2 * v + 1].x = ct * acc[2 * v + 1].x + (hx * u.x - hy * u.y - hz * d.x);
                    nx[2 * v + 1].y = ct * acc[2 * v + 1].y + (hx * u.y + hy * u.x - hz * d.y);
                }
            }
            if (m > 1) {
#pragma unroll
                for (int k = 0; k < 4; ++k) { const double2 pv = nxt[k * N + ii]; nx[k].x -= pv.x; nx[k].y -= pv.y; }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) nxt[k * N + ii] = nx[k];
            // Gram sums of this site (same definitions as cheb_step.cuh)
            if (MODE == kModeHund2) {
                gs[0] += nx[0].x * nx[0].x + nx[0].y * nx[0].y + nx[1].x * nx[1].x + nx[1].y * nx[1].y;
                gs[1] += nx[2].x * nx[2].x + nx[2].y * nx[2].y + nx[3].x * nx[3].x + nx[3].y * nx[3].y;
                gs[2] += nx[0].x * nx[2].x + nx[0].y * nx[2].y + nx[1].x * nx[3].x + nx[1].y * nx[3].y;
                gs[3] += nx[0].x * nx[2].y - nx[0].y * nx[2].x + nx[1].x * nx[3].y - nx[1].y * nx[3].x;
                gs[4] += c0[0].x * nx[0].x + c0[0].y * nx[0].y + c0[1].x * nx[1].x + c0[1].y * nx[1].y;
                gs[5] += c0[2].x * nx[2].x + c0[2].y * nx[2].y + c0[3].x * nx[3].x + c0[3].y * nx[3].y;
                gs[6] += c0[0].x * nx[2].x + c0[0].y * nx[2].y + c0[1].x * nx[3].x + c0[1].y * nx[3].y;
                gs[7] += c0[0].x * nx[2].y - c0[0].y * nx[2].x + c0[1].x * nx[3].y - c0[1].y * nx[3].x;
            } else if (MODE == kModeDex) {
                // per site q of the slot, start vectors o = chunk 2q, v = chunk 2q+1: (Yoo, Yvv, Re Yov, Im Yov, Xoo, Xvv, Re Xov, Im Xov)
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const double2 o = nx[2 * q], v = nx[2 * q + 1], op = c0[2 * q], vp = c0[2 * q + 1];
                    gs[8 * q + 0] += o.x * o.x + o.y * o.y;
                    gs[8 * q + 1] += v.x * v.x + v.y * v.y;
                    gs[8 * q + 2] += o.x * v.x + o.y * v.y;
                    gs[8 * q + 3] += o.x * v.y - o.y * v.x;
                    gs[8 * q + 4] += op.x * o.x + op.y * o.y;
                    gs[8 * q + 5] += vp.x * v.x + vp.y * v.y;
                    gs[8 * q + 6] += op.x * v.x + op.y * v.y;
                    gs[8 * q + 7] += op.x * v.y - op.y * v.x;
                }
            } else {
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const double2 u = nx[2 * q], d = nx[2 * q + 1], up = c0[2 * q], dp = c0[2 * q + 1];
                    gs[4 * q + 0] += u.x * u.x + u.y * u.y + d.x * d.x + d.y * d.y;
                    gs[4 * q + 1] += up.x * u.x + up.y * u.y + dp.x * d.x + dp.y * d.y;
                    gs[4 * q + 2] += gam[j] * (up.x * d.x - up.y * d.y - dp.x * u.x + dp.y * u.y);
                    gs[4 * q + 3] += gam[j] * (up.x * d.y + up.y * d.x - dp.x * u.y - dp.y * u.x);
                }
            }
        }
        // per-step reduction: warp (9 shuffles per 8 sums) -> shared memory -> the warps of a slot in index order; double-buffered by step parity
        double* rd = red + (size_t)(m & 1) * kResWarps * 16;
#pragma unroll
        for (int h = 0; h < NG / 8; ++h) {
            double part[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) part[k] = gs[8 * h + k];
            const double s = warp_reduce8(part, lane);
            if ((lane & 3) == 0) rd[warp * 16 + 8 * h + (lane >> 2)] = s;
        }
        __syncthreads();                 // also the step barrier: r_m complete, r_{m-1} no longer read
        if (tid < NG * G) {
            const int gg = tid / NG, k = tid % NG;
            const int sl = blockIdx.x * G + gg;
            if (sl < a.Ps) {
                double tot = 0.0;
                for (int w = gg * wps; w < (gg + 1) * wps; ++w) tot += rd[w * 16 + k];
                a.gram[((size_t)(m - 1) * a.Ps + sl) * NG + k] = tot;
            }
        }
    }
}

}  // namespace gfmc
