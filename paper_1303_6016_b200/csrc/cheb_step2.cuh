// cheb_step2.cuh -- TWO Chebyshev steps per pass over the work vectors (temporal blocking),
// for the one-vector mode of Eq. (1) (`ph_symmetry = 1`) on the 32^3 lattice, hand-written for sm_100a.
//
// One launch applies Eq. (26) twice,
//     r_m     = 2 H~ r_{m-1} - r_{m-2}        (first pass: r_1 = H~ r_0)
//     r_{m+1} = 2 H~ r_m     - r_{m-1},
// reading r_{m-1}, r_{m-2} from HBM once and writing r_m, r_{m+1} once: 64 B per complex element and TWO steps instead of
// 2 x 48 B.  r_m never comes back from HBM inside the pass: its planes live in a shared-memory ring between the two stencil stages.
//
//  * Layout of the four work buffers (the pass cannot run in place: a neighbouring CTA still needs the old rows):
//        R[z][p][y][s][x],  p = site of the batch (ONE start vector |o_p up> per site), s = spin component,
//    so that a y-slab of one site's plane is one contiguous range (1 KiB per row) for 1-D bulk TMA.
//  * Work item = (site p, y-tile of 16 rows), z-march over the whole column.  576 threads = 18 warps, lane = x:
//      stage 1: warp w computes r_m on row y0-1+w of plane t (18 rows: the tile plus one halo row on each side, recomputed
//               rather than exchanged) from r_{m-1} planes t-1, t, t+1 (bulk-TMA ring, 20 rows) and r_{m-2} (ring, 18 rows),
//               writes it to the r_m ring (shared memory) and, for the 16 interior rows, to HBM;
//      __syncthreads (the only barrier of a plane iteration);
//      stage 2: warps 1..16 compute r_{m+1} on plane t-1 from r_m planes t-2 (own site), t-1 (lateral neighbours; shared memory) and
//               t (own site: stage 1's result, still in registers) and r_{m-1}[t-1] (own site, carried in registers), and write it to HBM.
//    Planes t = -1 and t = L of r_m are recomputed as well (periodic z halo of stage 2).  Redundant work: 18/16 rows x 34/32 planes
//    of stage 1; redundant loads: 20/16 rows of r_{m-1}, 18/16 of r_{m-2} (L2 hits where the neighbouring tile runs alongside).
//  * All warps advance in lockstep through the one barrier per plane, so ring stages are recycled without empty-barriers: after the
//    barrier of iteration t plane t-2 of r_{m-1} and plane t of r_{m-2} are dead and thread 0 refills them (the loads run ahead
//    across work items).
//  * Gram sums of BOTH steps (Y, X, Re W, Im W per site and step) accumulate in registers over the interior rows and
//    planes only; one deterministic partial per (site, y-tile, step).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "cheb_step.cuh"

namespace gfmc {

constexpr int k2L = 32;                    // lattice edge served by this kernel
constexpr int k2Ty = 16;                   // interior rows of a tile
constexpr int k2Warps = k2Ty + 2;          // one warp per stage-1 row
constexpr int k2Threads = 32 * k2Warps;    // 576
constexpr int k2RowU = 2 * k2L;            // double2 per row of one site's plane: 2 spin components x 32
constexpr int k2CurRows = k2Ty + 4, k2MidRows = k2Ty + 2;
// Ring depths: r_{m-1} (bulk TMA; planes t and t+1 are live in an iteration), r_m (produced here: plane t is written while t-1 is read
// laterally and t-2 at the own site), r_{m-2} (bulk TMA, one plane live).  Same-box sweep at config 4 (site updates/s, 2 repetitions,
// scatter 0.3 %): (NC, NP) = (4,3) 4335, (4,5) 4312, (5,3) 4121, (5,2) 4103, (3,4) 4088, (3,3) 4075, (4,4) 3808, (6,1) 2604.
constexpr int k2NC = 4, k2NM = 3, k2NP = 3;
constexpr int k2CurU = k2CurRows * k2RowU, k2MidU = k2MidRows * k2RowU;
constexpr int k2HeaderBytes = 2048;
constexpr size_t k2SmemBytes = k2HeaderBytes + (size_t)16 * (k2NC * k2CurU + k2NM * k2MidU + k2NP * k2MidU);

struct Step2Args {
    const double2* cur;      // r_{m-1}
    const double2* prv;      // r_{m-2} (ignored in the first pass)
    double2* out1;           // r_m
    double2* out2;           // r_{m+1}
    const double* Sx; const double* Sy; const double* Sz;
    double* gram1;           // Gram partials of step m  : [Pslots][2 tiles][8], entry 4*(p&1) + k of slot p>>1 (layout of finalize_moments_ph)
    double* gram2;           // Gram partials of step m+1
    double ct1, cj1;         // -scale t/a, scale J_H/a of the first step of the pass (scale = 1 in the first pass, else 2)
    double ct2, cj2;         // same for the second step (scale = 2)
    int P;                   // sites (= start vectors) in this launch
    int nitems;              // 2 P
};

struct Step2Header {
    uint64_t full_c[k2NC], full_p[k2NP];
    double red[k2Warps * 8];
};
static_assert(sizeof(Step2Header) <= k2HeaderBytes, "header too large");

// next load of a ring in consumption order: (item, plane q); r_{m-1}: q = -2 .. L+1, r_{m-2}: q = -1 .. L
struct Load2Cursor { int item, q; };

__device__ __forceinline__ void step2_issue_cur(const Step2Args& a, Load2Cursor& cu, uint64_t* full, double2* dst)
{
    constexpr int L = k2L;
    const int p = cu.item >> 1, y0 = (cu.item & 1) * k2Ty;
    const int z = (cu.q + L) % L;
    const double2* plane = a.cur + ((size_t)z * a.P + p) * L * k2RowU;
    mbar_arrive_expect_tx(full, k2CurRows * k2RowU * 16u);
    // rows y0-2 .. y0+17 (periodic): two contiguous pieces
    if (y0 == 0) {
        bulk_g2s(dst, plane + (size_t)(L - 2) * k2RowU, 2u * k2RowU * 16u, full);
        bulk_g2s(dst + 2 * k2RowU, plane, (uint32_t)(k2CurRows - 2) * k2RowU * 16u, full);
    } else {
        bulk_g2s(dst, plane + (size_t)(y0 - 2) * k2RowU, (uint32_t)(k2CurRows - 2) * k2RowU * 16u, full);
        bulk_g2s(dst + (size_t)(k2CurRows - 2) * k2RowU, plane, 2u * k2RowU * 16u, full);
    }
    if (++cu.q > L + 1) { cu.q = -2; cu.item += gridDim.x; }
}

__device__ __forceinline__ void step2_issue_prv(const Step2Args& a, Load2Cursor& cu, uint64_t* full, double2* dst)
{
    constexpr int L = k2L;
    const int p = cu.item >> 1, y0 = (cu.item & 1) * k2Ty;
    const int z = (cu.q + L) % L;
    const double2* plane = a.prv + ((size_t)z * a.P + p) * L * k2RowU;
    mbar_arrive_expect_tx(full, k2MidRows * k2RowU * 16u);
    // rows y0-1 .. y0+16 (periodic)
    if (y0 == 0) {
        bulk_g2s(dst, plane + (size_t)(L - 1) * k2RowU, k2RowU * 16u, full);
        bulk_g2s(dst + k2RowU, plane, (uint32_t)(k2MidRows - 1) * k2RowU * 16u, full);
    } else {
        bulk_g2s(dst, plane + (size_t)(y0 - 1) * k2RowU, (uint32_t)(k2MidRows - 1) * k2RowU * 16u, full);
        bulk_g2s(dst + (size_t)(k2MidRows - 1) * k2RowU, plane, k2RowU * 16u, full);
    }
    if (++cu.q > L) { cu.q = -1; cu.item += gridDim.x; }
}

// (h.sigma)(u, d)^T + ct * acc  for one site: up = hz u + (hx - i hy) d, down = (hx + i hy) u - hz d
__device__ __forceinline__ void step2_apply(double ct, double hx, double hy, double hz, const double2 (&acc)[2], const double2 (&c)[2], double2 (&nx)[2])
{
    const double2 u = c[0], d = c[1];
    nx[0].x = ct * acc[0].x + (hz * u.x + hx * d.x + hy * d.y);
    nx[0].y = ct * acc[0].y + (hz * u.y + hx * d.y - hy * d.x);
    nx[1].x = ct * acc[1].x + (hx * u.x - hy * u.y - hz * d.x);
    nx[1].y = ct * acc[1].y + (hx * u.y + hy * u.x - hz * d.y);
}

// (Y, X, Re W, Im W) of one site for the pair (older = r_{k-1}, newer = r_k) -- DESIGN.md §5.3; gam = Gamma_i = (-1)^(x+y+z)
__device__ __forceinline__ void step2_gram(double (&g)[4], const double2 (&older)[2], const double2 (&newer)[2], double gam)
{
    const double2 u = newer[0], d = newer[1], up = older[0], dp = older[1];
    g[0] += u.x * u.x + u.y * u.y + d.x * d.x + d.y * d.y;
    g[1] += up.x * u.x + up.y * u.y + dp.x * d.x + dp.y * d.y;
    g[2] += gam * (up.x * d.x - up.y * d.y - dp.x * u.x + dp.y * u.y);
    g[3] += gam * (up.x * d.y + up.y * d.x - dp.x * u.y - dp.y * u.x);
}

template <bool FIRST>
__global__ void __launch_bounds__(k2Threads, 1) cheb_step2_kernel(const __grid_constant__ Step2Args a)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    Step2Header* hdr = reinterpret_cast<Step2Header*>(smem_raw);
    double2* ring_c = reinterpret_cast<double2*>(smem_raw + k2HeaderBytes);
    double2* ring_m = ring_c + (size_t)k2NC * k2CurU;
    double2* ring_p = ring_m + (size_t)k2NM * k2MidU;

    constexpr int L = k2L;
    const int tid = threadIdx.x, w = tid >> 5, x = tid & 31;
    const int xm = (x + L - 1) & (L - 1), xp = (x + 1) & (L - 1);
    const bool interior = (w >= 1 && w <= k2Ty);

    Load2Cursor cu_c{(int)blockIdx.x, -2}, cu_p{(int)blockIdx.x, -1};     // thread 0's copies are the live ones
    uint32_t issued_c = 0, issued_p = 0;                                  // loads issued so far (thread 0)
    if (tid == 0) {
        for (int s = 0; s < k2NC; ++s) mbar_init(&hdr->full_c[s], 1);
        for (int s = 0; s < k2NP; ++s) mbar_init(&hdr->full_p[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        for (int s = 0; s < k2NC && cu_c.item < a.nitems; ++s, ++issued_c)
            step2_issue_cur(a, cu_c, &hdr->full_c[s], ring_c + (size_t)s * k2CurU);
        if (!FIRST)
            for (int s = 0; s < k2NP && cu_p.item < a.nitems; ++s, ++issued_p)
                step2_issue_prv(a, cu_p, &hdr->full_p[s], ring_p + (size_t)s * k2MidU);
    }
    __syncthreads();

    uint32_t nc = 0, np = 0, nm = 0;     // planes consumed so far from the r_{m-1} ring / r_{m-2} ring; r_m planes produced so far
    // refill after a barrier: `dead` planes of a ring have been retired since the kernel started
    auto refill = [&](uint32_t dead_c, uint32_t dead_p) {
        if (tid == 0) {
            // generic-proxy reads of the retired stages (all warps, ordered by the barrier) before the async-proxy writes of the refill
            fence_proxy_async_shared();
            while (issued_c < dead_c + k2NC && cu_c.item < a.nitems) {
                const uint32_t s = issued_c % k2NC;
                step2_issue_cur(a, cu_c, &hdr->full_c[s], ring_c + (size_t)s * k2CurU);
                ++issued_c;
            }
            if (!FIRST)
                while (issued_p < dead_p + k2NP && cu_p.item < a.nitems) {
                    const uint32_t s = issued_p % k2NP;
                    step2_issue_prv(a, cu_p, &hdr->full_p[s], ring_p + (size_t)s * k2MidU);
                    ++issued_p;
                }
        }
    };

    for (int item = blockIdx.x; item < a.nitems; item += gridDim.x) {
        const int p = item >> 1, y0 = (item & 1) * k2Ty;
        const int y1 = (y0 - 1 + w + L) & (L - 1);              // row of this warp in stage 1 (and, for interior warps, in stage 2)
        const int site_xy = x + L * y1;
        double g1[4] = {0, 0, 0, 0}, g2[4] = {0, 0, 0, 0};
        // Spins of the column (x, y1): loaded ONE ITERATION AHEAD of their first use (L2 hits, but ~1 us away: consumed directly they were
        // the top stall of the first version, 26 % of all warp samples); stage 1 works on plane t with (sx, sy, sz), stage 2 on plane t-1
        // with the set stage 1 used one iteration earlier.
        double sx_o = 0, sy_o = 0, sz_o = 0;
        double sx_n, sy_n, sz_n;
        {
            const int si0 = site_xy + L * L * (L - 1);          // plane t = -1
            sx_n = __ldg(a.Sx + si0); sy_n = __ldg(a.Sy + si0); sz_n = __ldg(a.Sz + si0);
        }
        double2* out1 = a.out1 + ((size_t)p * L + y1) * k2RowU + x;      // + z * zstride
        double2* out2 = a.out2 + ((size_t)p * L + y1) * k2RowU + x;
        const size_t zstride = (size_t)a.P * L * k2RowU;

        // planes -2 and -1 of r_{m-1}
        const uint32_t c_base = nc;                             // ring index of plane q is c_base + (q + 2)
        mbar_wait(&hdr->full_c[c_base % k2NC], (c_base / k2NC) & 1u);
        mbar_wait(&hdr->full_c[(c_base + 1) % k2NC], ((c_base + 1) / k2NC) & 1u);
        const uint32_t p_base = np, m_base = nm;                // r_{m-2} plane q: p_base + (q + 1); r_m plane q: m_base + (q + 1)
        // Carried in registers from one iteration to the next (8 of the 32 shared-memory reads of an iteration):
        //   cprev = r_{m-1} of this site at plane t-1 (stage 1's lower z neighbour AND the "- r_{m-1}" of stage 2),
        //   nxp   = r_m of this site at plane t-1 (stage 2's centre); r_m at plane t is stage 1's own result.
        double2 cprev[2], nxp[2];
        {
            const double2* c2 = ring_c + (size_t)(c_base % k2NC) * k2CurU + (w + 1) * k2RowU;            // plane -2
#pragma unroll
            for (int s = 0; s < 2; ++s) { cprev[s] = c2[s * L + x]; nxp[s] = make_double2(0.0, 0.0); }
        }

        for (int t = -1; t <= L; ++t) {
            // Both stages of an iteration are ONE straight-line block between two barriers: stage 2 (plane t-1) needs nothing that OTHER warps
            // produce in stage 1 of this iteration (r_m of plane t enters only at the own site, i.e. from this thread's registers; the
            // lateral r_m neighbours are plane t-1, written one iteration earlier), so the two instruction streams are independent and
            // the waits sit in front of them, the global stores behind them.
            const uint32_t ic = c_base + (uint32_t)(t + 2);     // ring index of plane t of r_{m-1}; t+1: ic+1
            mbar_wait(&hdr->full_c[(ic + 1) % k2NC], ((ic + 1) / k2NC) & 1u);
            const uint32_t ip = p_base + (uint32_t)(t + 1);
            if (!FIRST) mbar_wait(&hdr->full_p[ip % k2NP], (ip / k2NP) & 1u);
            const double2* c0 = ring_c + (size_t)(ic % k2NC) * k2CurU;
            const double2* cp = ring_c + (size_t)((ic + 1) % k2NC) * k2CurU;
            const int rc = (w + 1) * k2RowU;                    // this warp's row inside an r_{m-1} stage (row 0 = y0-2)
            const double sx = sx_n, sy = sy_n, sz = sz_n;
            {
                const int si = site_xy + L * L * ((t + 1) & (L - 1));      // plane t+1 (unused after the last iteration)
                sx_n = __ldg(a.Sx + si); sy_n = __ldg(a.Sy + si); sz_n = __ldg(a.Sz + si);
            }
            // ---------------------------------------------------------------- stage 1: r_m on plane t, row y1
            double2 acc[2], cc[2], nx[2];
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int o = rc + s * L;
                acc[s] = add2(add2(add2(cprev[s], cp[o + x]), add2(c0[o + xm], c0[o + xp])), add2(c0[o - k2RowU + x], c0[o + k2RowU + x]));
                cc[s] = c0[o + x];
            }
            step2_apply(a.ct1, a.cj1 * sx, a.cj1 * sy, a.cj1 * sz, acc, cc, nx);
            if (!FIRST) {
                const double2* pv = ring_p + (size_t)(ip % k2NP) * k2MidU + w * k2RowU;
#pragma unroll
                for (int s = 0; s < 2; ++s) { const double2 v = pv[s * L + x]; nx[s].x -= v.x; nx[s].y -= v.y; }
            }
            const uint32_t im1 = m_base + (uint32_t)(t + 1);    // ring index of plane t of r_m; t-1: im1-1; t-2: im1-2
            {
                double2* md = ring_m + (size_t)(im1 % k2NM) * k2MidU + w * k2RowU;
#pragma unroll
                for (int s = 0; s < 2; ++s) md[s * L + x] = nx[s];
            }
            const bool store1 = interior && t >= 0 && t < L;
            if (store1) step2_gram(g1, cc, nx, ((x + y1 + t) & 1) ? -1.0 : 1.0);

            // ---------------------------------------------------------------- stage 2: r_{m+1} on plane k = t-1, interior rows
            const int k = t - 1;
            const bool store2 = interior && k >= 0;
            double2 nx2[2];
            if (store2) {
                const double2* mm = ring_m + (size_t)((im1 - 2) % k2NM) * k2MidU;     // plane t-2: own site only
                const double2* m0 = ring_m + (size_t)((im1 - 1) % k2NM) * k2MidU;     // plane t-1: lateral neighbours (written one iteration ago)
                const int rm = w * k2RowU;
                double2 acc2[2];
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const int o = rm + s * L;
                    acc2[s] = add2(add2(add2(mm[o + x], nx[s]), add2(m0[o + xm], m0[o + xp])), add2(m0[o - k2RowU + x], m0[o + k2RowU + x]));
                }
                step2_apply(a.ct2, a.cj2 * sx_o, a.cj2 * sy_o, a.cj2 * sz_o, acc2, nxp, nx2);
#pragma unroll
                for (int s = 0; s < 2; ++s) { nx2[s].x -= cprev[s].x; nx2[s].y -= cprev[s].y; }     // - r_{m-1} of this site at plane t-1
                step2_gram(g2, nxp, nx2, ((x + y1 + k) & 1) ? -1.0 : 1.0);
            }
            // ---------------------------------------------------------------- global stores of both stages
            if (store1) {
#pragma unroll
                for (int s = 0; s < 2; ++s) stg_stream(out1 + (size_t)t * zstride + s * L, nx[s]);
            }
            if (store2) {
#pragma unroll
                for (int s = 0; s < 2; ++s) stg_stream(out2 + (size_t)k * zstride + s * L, nx2[s]);
            }
            sx_o = sx; sy_o = sy; sz_o = sz;
#pragma unroll
            for (int s = 0; s < 2; ++s) { cprev[s] = cc[s]; nxp[s] = nx[s]; }
            __syncthreads();
            // Plane t of r_{m-1} is dead: stage 1 of iteration t was its only reader (lateral neighbours and centre; the own-site values
            // that later stages still need travel in registers), and so is plane t of r_{m-2}.
            refill(c_base + (uint32_t)(t + 3), p_base + (uint32_t)(t + 2));
        }
        nc += L + 4; np += L + 2; nm += L + 2;

        // ---------------------------------------------------------- per-item reduction of the 2 x 4 Gram sums (interior warps, fixed order)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                g1[q] += __shfl_xor_sync(0xffffffffu, g1[q], off);
                g2[q] += __shfl_xor_sync(0xffffffffu, g2[q], off);
            }
        }
        if (x == 0) {
#pragma unroll
            for (int q = 0; q < 4; ++q) { hdr->red[w * 8 + q] = g1[q]; hdr->red[w * 8 + 4 + q] = g2[q]; }
        }
        __syncthreads();
        // every stage-2 read of this item is behind the barrier: planes L-1, L, L+1 of r_{m-1} are dead too
        refill(nc, np);
        if (tid < 8) {
            double sacc = 0.0;
            for (int ww = 1; ww <= k2Ty; ++ww) sacc += hdr->red[ww * 8 + tid];
            double* dst = (tid < 4 ? a.gram1 : a.gram2) + ((size_t)(p >> 1) * 2 + (item & 1)) * 8 + 4 * (p & 1) + (tid & 3);
            *dst = sacc;
        }
        __syncthreads();
    }
}

// |r_0> = |o_p up> in the layout R[z][p][y][s][x] (the buffer has been zeroed)
__global__ void init_start_vectors_ph2(double2* R0, const int32_t* __restrict__ sites, int P, int L)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    const int o = sites[p];
    const int x = o % L, y = (o / L) % L, z = o / (L * L);
    R0[(((size_t)z * P + p) * L + y) * 2 * L + x] = make_double2(1.0, 0.0);
}

}  // namespace gfmc
