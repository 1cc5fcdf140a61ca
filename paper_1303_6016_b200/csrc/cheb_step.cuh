// cheb_step.cuh -- the fused Chebyshev step, hand-written for sm_100a.
//
// One launch performs ONE application of the three-term recursion of Eq. (26)
//     r_{m} = 2 H~ r_{m-1} - r_{m-2}        (first step: r_1 = H~ r_0)
// to ALL start vectors of a batch, with H of Eq. (1) applied matrix-free (6-neighbour
// periodic stencil + 2x2 on-site Hund block from the spin field), and accumulates, in registers, the
// two Gram blocks that Eq. (27)-(28) turn into the moments mu_{2m-1}, mu_{2m}:
//     Y(a,b) = <r^a_m | r^b_m>,   X(a,b) = <r^a_{m-1} | r^b_m>,   a,b in {up,down start vector of one site}.
//
// The paper's own kernel ("CalculateCoefficient": ELLPACK SpMV, one row per thread, one
// vector at a time, shared-memory block reduction) is prior art; this design differs:
//
//  * Data layout in HBM (work vectors R_cur / R_prev, complex fp64 = double2):
//        R[z][p][y][c][x],  p = pair (= site being updated) of the batch,  c = 2*vi + s
//    vi = which start vector of the pair (0: |o up>, 1: |o down>), s = spin component of the element.
//    A whole xy-plane of one pair (or a y-slab of it) is ONE contiguous byte range -> moved by 1-D bulk
//    TMA (cp.async.bulk, SASS UBLKCP) with no tensor map; a warp reading one chunk-row reads 512
//    contiguous bytes (32 lanes x 16 B) from shared or global memory, conflict-free.
//  * Persistent CTAs (one per SM, 16 warps, all consumers) walk a list of work items (pair-group, y-tile,
//    z-chunk) and march along z.  R_cur planes (slab + 2 halo rows) stream through a CTA-wide shared-memory
//    ring by bulk TMA; a stage is refilled by whichever warp releases it last ("ring refill" below), so the
//    prefetch runs ahead across work items and nobody blocks on an empty stage.  r_{m-2} (R_prev) is private
//    to the thread that overwrites it: for compile-time L every warp streams its own 2 KiB segment through a
//    private ring (warp_prev_issue).  The 512 threads own one lattice site each (all 4 chunks: both start
//    vectors x both spin components), carry the z-1 column in registers, read the z / z+1 columns and the 4
//    lateral neighbours from the ring, and write r_m to global memory with 128-bit streaming stores (in place
//    over r_{m-2}).
//  * The Hund term and all 8 Gram sums are thread-local (no shuffles in the plane loop); one warp-shuffle +
//    shared-memory reduction per work item writes a deterministic partial per (pair, tile).
//  * No tensor cores: the path is a stencil at ~1.3 flop/B, HBM-bound.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gfmc {

constexpr int kConsumerThreads = 512;
constexpr int kConsumerWarps = kConsumerThreads / 32;
constexpr int kStepThreads = kConsumerThreads;
constexpr int kMaxStages = 8;
constexpr int kMaxWarpStages = 4;         // depth limit of the per-warp R_prev rings
constexpr int kWarpSegUnits = 128;        // double2 per per-warp R_prev stage: 32 sites x 4 chunks = 2 KiB

// What the 4 chunks of a slot p hold, and which Gram sums a step accumulates (DESIGN.md §5.1 "modes"):
//  kModeHund2: Eq. (1), slot = one site o, chunk c = 2*vi + s: both start vectors |o up>, |o dn> (the definition of row a3).
//  kModeHund1: Eq. (1), slot = TWO sites, chunk c = 2*q + s: only |o_q up> is propagated; |o_q dn>'s vector follows from the
//              antiunitary symmetry A = Gamma (i sigma_y) K, A H A^-1 = -H on an even-L (bipartite) lattice.
//  kModeDex  : Eq. (2)-(3) (J_H -> inf), one orbital per site, slot = TWO sites, chunk c = 2*q + vi: start vectors |o_q>, |v_q>
//              of Eq. (21); complex bond amplitudes instead of the on-site Hund block.
constexpr int kModeHund2 = 0, kModeHund1 = 1, kModeDex = 2;
__host__ __device__ constexpr int gram_width(int mode) { return mode == kModeDex ? 16 : 8; }

struct StepArgs {
    const double2* cur;      // R_cur  : r_{m-1}, read-only in this launch
    double2*       nxt;      // R_prev : r_{m-2} on entry (ignored when FIRST), r_m on exit (in place)
    const double*  Sx;       // spin field, SoA [N]
    const double*  Sy;
    const double*  Sz;
    const double2* Tx;       // kModeDex only: forward bond amplitudes t_{i,i+e_d} of Eq. (3), SoA [N] per direction
    const double2* Ty;
    const double2* Tz;
    const double2* Tq;       // kModeDex only: the same amplitudes interleaved per lattice row, T[z][y][d][x], d = (z, x, y) bond: the rows a warp
                             // needs in one plane are one contiguous range (per-warp bond rings below)
    double*        gram;     // partial Gram sums of this step: [P][ntiles][NG], NG = gram_width(MODE)
    double ct;               // hopping coefficient: -scale*t/a   (scale = 1 first step, 2 afterwards)
    double cj;               // Hund coefficient:     scale*J_H/a
    int L, P;                // lattice edge, pairs in this launch
    int full;                // 1: a CTA tile is G whole xy-planes (small L); 0: a y-slab of Ty rows of one pair + 2 halo rows
    int G, Ty_rows, nty, nzc, nzper;
    int nitems;              // npg * nzc * nty
    int nst_c, nst_p;        // ring depths: R_cur ring, R_prev ring
    int nst_t;               // depth of the per-warp bond-amplitude rings (kModeDex with compile-time L <= 32; 0: amplitudes come by ld.global.nc)
    int tstage_units;        // double2 per bond stage of the whole CTA: kConsumerWarps * (3 * rows per warp + 1) * L
    int cstage_units;        // double2 per R_cur stage  (rows incl. halo) * 4L
    int pstage_units;        // double2 per R_prev stage (rows)            * 4L
    int slow_reduce;         // 1: sites per pair in a tile is not a multiple of 32 (odd L): generic reduction
    // Optional explicit work list ("stream-K" decomposition, see make_item_table in gfmc_api.cu): CTA b processes
    // items[cta_start[b] .. cta_start[b+1]) in order.  Every CTA gets the same number of planes; a (pair group, y-tile) column that
    // straddles two CTAs is cut in z (each piece re-reads its two halo planes).  nullptr: items are enumerated arithmetically
    // (item = blockIdx.x + k * gridDim.x, z chunks of nzper planes).
    const struct WorkItem* items;
    const int* cta_start;
    int ntiles;              // Gram partials per pair and step (nty * nzc, or nty * 2 with the explicit list)
};
struct WorkItem { int pg, ty, z0, nz, tile; };

// ---------------------------------------------------------------- PTX helpers (mbarrier + bulk TMA)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// non-blocking: has the phase of parity `parity` completed?  (acquire.cta by default)
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ uint32_t cas_relaxed_shared(uint32_t* p, uint32_t expect, uint32_t desired) {
    uint32_t old;
    asm volatile("atom.relaxed.cta.shared.cas.b32 %0, [%1], %2, %3;" : "=r"(old) : "r"(smem_u32(p)), "r"(expect), "r"(desired) : "memory");
    return old;
}
// 1-D bulk copy global -> shared, completion signalled on an mbarrier (TMA, SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// barrier among the consumer warps only (the producer warp never joins it)
__device__ __forceinline__ void consumer_bar_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kConsumerThreads) : "memory"); }
// streaming 128-bit global store for r_m (touched exactly once per launch)
__device__ __forceinline__ void stg_stream(double2* p, double2 v) {
    asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// orders this thread's earlier generic-proxy accesses to shared memory before later async-proxy (bulk TMA) writes to it
__device__ __forceinline__ void fence_proxy_async_shared() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ double2 add2(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }

// shared memory carve-up: [barriers][reduction scratch] | R_cur ring | R_prev ring | (slow reduction scratch)
struct StepSmemHeader {
    uint64_t full_c[kMaxStages], full_p[kMaxStages];          // TMA completion barriers
    uint64_t empty_c[kMaxStages];                             // R_cur ring: "all 16 warps are done with the stage" barriers
    uint32_t seq_c[kMaxStages];                               // R_cur ring: number of refills issued into the stage (dedupes the refill)
    uint32_t rel_p[kMaxStages];                               // R_prev ring (run-time L only): release counters (0 .. kConsumerWarps)
    int      cur_item, cur_q, prev_item, prev_q;              // refill cursors (RingCursor x 2)
    uint64_t full_w[kConsumerWarps][kMaxWarpStages];          // per-warp rings (compile-time L): TMA completion barriers; R_prev stages first,
                                                              // then the bond-amplitude stages (nst_p + nst_t <= kMaxWarpStages)
    double   red[kConsumerWarps * 16];    // fast reduction: one row of NG <= 16 sums per consumer warp
};
constexpr int kStepHeaderBytes = 3072;    // header padded so that ring stages are 1 KiB aligned
static_assert(sizeof(StepSmemHeader) <= kStepHeaderBytes, "header too large");

struct ItemCoord { int pg, ty, zc, z0, nz, y0, rows; };      // zc: z-chunk index, or (explicit work list) the Gram tile index

template <bool SK>
__device__ __forceinline__ ItemCoord decode_item(const StepArgs& a, int item) {
    ItemCoord c;
    if (SK) {
        const WorkItem w = a.items[item];
        c.pg = w.pg; c.ty = w.ty; c.z0 = w.z0; c.nz = w.nz; c.zc = w.tile;
    } else {
        c.ty = item % a.nty;
        int rest = item / a.nty;
        c.zc = rest % a.nzc;
        c.pg = rest / a.nzc;
        c.z0 = c.zc * a.nzper;
        c.nz = min(a.nzper, a.L - c.z0);
    }
    c.y0 = c.ty * a.Ty_rows;
    c.rows = a.full ? a.L : min(a.Ty_rows, a.L - c.y0);
    return c;
}

// the item sequence of this CTA: first index, end (exclusive), stride
template <bool SK> __device__ __forceinline__ int item_first(const StepArgs& a) { return SK ? a.cta_start[blockIdx.x] : (int)blockIdx.x; }
template <bool SK> __device__ __forceinline__ int item_end(const StepArgs& a) { return SK ? a.cta_start[blockIdx.x + 1] : a.nitems; }
template <bool SK> __device__ __forceinline__ int item_stride(const StepArgs& a) { return SK ? 1 : (int)gridDim.x; }

// ------------------------------------------------------------------ ring refill ("last releaser issues")
// There is no producer warp and nobody ever blocks on an empty stage: every consumer warp releases a stage by
// bumping that stage's counter (acq_rel); the warp whose bump is the 16th knows that every warp is done with the
// stage and immediately issues the next bulk-TMA load of that ring into it.  Loads of a ring are issued in
// consumption order (stages are released in order), so "the next load" is a cursor (item, q) kept in shared
// memory and touched only by the current last releaser.  R_cur: planes q = -1 .. nz of every item (nz + 2 loads,
// slab + 2 halo rows each); R_prev: planes q = 0 .. nz-1.
struct RingCursor { int item, q; };

__device__ __forceinline__ uint32_t atom_add_acq_rel_shared(uint32_t* p, uint32_t v) {
    uint32_t old;
    asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(smem_u32(p)), "r"(v) : "memory");
    return old;
}

template <int LT, bool SK>
__device__ __noinline__ void issue_cur(const StepArgs& a, RingCursor* cu, uint64_t* full, double2* dst)
{
    const int L = LT ? LT : a.L;
    const int rowu = 4 * L;
    int item = cu->item, q = cu->q;
    if (item >= item_end<SK>(a)) return;
    const ItemCoord c = decode_item<SK>(a, item);
    const int p0 = c.pg * a.G;
    const int zq = (c.z0 + q + L) % L;
    const double2* pp = a.cur + ((size_t)zq * a.P + p0) * L * rowu;
    if (a.full) {
        const uint32_t bytes = (uint32_t)min(a.G, a.P - p0) * L * rowu * 16u;
        mbar_arrive_expect_tx(full, bytes);
        bulk_g2s(dst, pp, bytes, full);
    } else {
        const uint32_t rbytes = (uint32_t)rowu * 16u;
        const uint32_t mbytes = (uint32_t)c.rows * rbytes;
        const int ylo = (c.y0 + L - 1) % L, yhi = (c.y0 + c.rows) % L;
        mbar_arrive_expect_tx(full, mbytes + 2u * rbytes);
        bulk_g2s(dst + rowu, pp + (size_t)c.y0 * rowu, mbytes, full);
        bulk_g2s(dst, pp + (size_t)ylo * rowu, rbytes, full);
        bulk_g2s(dst + (size_t)(c.rows + 1) * rowu, pp + (size_t)yhi * rowu, rbytes, full);
    }
    if (++q > c.nz) { q = -1; item += item_stride<SK>(a); }
    cu->item = item; cu->q = q;
}

template <int LT, bool SK>
__device__ __noinline__ void issue_prev(const StepArgs& a, RingCursor* cu, uint64_t* full, double2* dst)
{
    const int L = LT ? LT : a.L;
    const int rowu = 4 * L;
    int item = cu->item, q = cu->q;
    if (item >= item_end<SK>(a)) return;
    const ItemCoord c = decode_item<SK>(a, item);
    const int p0 = c.pg * a.G;
    const double2* pp = a.nxt + ((size_t)(c.z0 + q) * a.P + p0) * L * rowu;
    uint32_t bytes;
    if (a.full) bytes = (uint32_t)min(a.G, a.P - p0) * L * rowu * 16u;
    else { bytes = (uint32_t)c.rows * rowu * 16u; pp += (size_t)c.y0 * rowu; }
    mbar_arrive_expect_tx(full, bytes);
    bulk_g2s(dst, pp, bytes, full);
    if (++q >= c.nz) { q = 0; item += item_stride<SK>(a); }
    cu->item = item; cu->q = q;
}

// ------------------------------------------------------------------ per-warp R_prev rings (compile-time L only)
// r_{m-2} is private to the thread that overwrites it.  For L in {8,16,32,64} the 32 sites of a warp are 32/L whole rows
// (L <= 32: ONE contiguous 2 KiB range of R_prev) or a 32-wide x segment of one row (L = 64: four 512 B pieces), so every warp
// streams its own segment through its own small ring: no cross-warp release, no atomics, and the warp refills a stage the moment
// it has read it (the refill lands nst_p planes ahead of the warp's own position, independent of how far the other warps are).
// The warp keeps a cursor over ITS sequence of planes (all planes of every item of this CTA in which the warp has sites, in
// order): the common case -- the next plane of the same item -- is a pointer bump; only the step to the next item decodes.
struct WarpPrevCursor { const double2* src; int item; int left; };

template <int LT, bool SK>
__device__ __noinline__ WarpPrevCursor warp_prev_next_item(const StepArgs& a, int warp, int item)
{
    WarpPrevCursor cu;
    constexpr int L = LT ? LT : 32;
    constexpr int rowu = 4 * L;
    constexpr bool full_mode = L * L <= kConsumerThreads;
    constexpr int plane_sites = full_mode ? L * L : kConsumerThreads;
    for (;;) {
        item += item_stride<SK>(a);
        if (item >= item_end<SK>(a)) { cu.src = nullptr; cu.item = item_end<SK>(a); cu.left = 0; return cu; }
        const ItemCoord c = decode_item<SK>(a, item);
        int g = 0;
        bool act;
        if (full_mode) { g = (32 * warp) / plane_sites; act = (g < a.G) && (c.pg * a.G + g < a.P); }
        else act = (32 * warp) / L < c.rows;
        if (!act) continue;
        const int rem0 = 32 * warp - g * plane_sites;
        const int yl0 = rem0 / L, x0 = rem0 % L;
        const int p = c.pg * a.G + g;
        cu.src = a.nxt + (((size_t)c.z0 * a.P + p) * L + (c.y0 + yl0)) * rowu + x0;
        cu.item = item; cu.left = c.nz;
        return cu;
    }
}

// issue the next plane of the warp's sequence into stage `dst` (one lane calls this)
template <int LT, bool SK>
__device__ __forceinline__ void warp_prev_issue(const StepArgs& a, int warp, WarpPrevCursor& cu, size_t zstride, uint64_t* full, double2* dst)
{
    constexpr int L = LT ? LT : 32;
    if (cu.left == 0) {
        if (cu.item >= item_end<SK>(a)) return;
        cu = warp_prev_next_item<LT, SK>(a, warp, cu.item);
        if (cu.left == 0) return;
    }
    mbar_arrive_expect_tx(full, kWarpSegUnits * 16u);
    if (L <= 32) {
        bulk_g2s(dst, cu.src, kWarpSegUnits * 16u, full);
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) bulk_g2s(dst + 32 * k, cu.src + (size_t)k * L, 32u * 16u, full);
    }
    cu.src += zstride;
    --cu.left;
}

// ------------------------------------------------------------------ per-warp bond-amplitude rings (kModeDex, compile-time L <= 32)
// The six bond amplitudes of a site (Eq. (3)) are the same for every slot of the batch and small (48 B per site), but
// read by ld.global at the top of a plane iteration they sit on the critical path of the first stencil FMA (ncu, round 1:
// long_scoreboard 4.3 stalls per issue).  They are staged like r_{m-2}: in the interleaved table T[z][y][d][x] (d = z-, x-, y-bond)
// the forward bonds of the warp's 32/L rows plus the y-bond row below them -- whose entries are the warp's BACKWARD y bonds -- are one
// contiguous range of (3 * 32/L + 1) * L amplitudes (two pieces where row y-1 wraps), streamed by the warp through its own ring.
// The backward x bond is the left neighbour's forward bond in the same row (periodic in x inside the row), the backward z bond is
// the forward z bond the thread itself read one plane earlier (carried in registers).
struct WarpBondCursor { const double2* src; int item; int left; int wrap; };

template <int LT, bool SK>
__device__ __noinline__ WarpBondCursor warp_bond_next_item(const StepArgs& a, int warp, int item)
{
    WarpBondCursor cu;
    constexpr int L = LT ? LT : 32;
    constexpr bool full_mode = L * L <= kConsumerThreads;
    constexpr int plane_sites = full_mode ? L * L : kConsumerThreads;
    for (;;) {
        item += item_stride<SK>(a);
        if (item >= item_end<SK>(a)) { cu.src = nullptr; cu.item = item_end<SK>(a); cu.left = 0; cu.wrap = 0; return cu; }
        const ItemCoord c = decode_item<SK>(a, item);
        int g = 0;
        bool act;
        if (full_mode) { g = (32 * warp) / plane_sites; act = (g < a.G) && (c.pg * a.G + g < a.P); }
        else act = (32 * warp) / L < c.rows;
        if (!act) continue;
        const int y = c.y0 + (32 * warp - g * plane_sites) / L;
        cu.src = a.Tq + ((size_t)c.z0 * L + y) * 3 * L;      // first forward row of the warp at plane z0
        cu.item = item; cu.left = c.nz; cu.wrap = (y == 0);
        return cu;
    }
}

template <int LT, bool SK>
__device__ __forceinline__ void warp_bond_issue(const StepArgs& a, int warp, WarpBondCursor& cu, uint64_t* full, double2* dst)
{
    constexpr int L = LT ? LT : 32;
    constexpr int fwd = 3 * (32 / L) * L;                     // forward amplitudes of the warp's rows
    if (cu.left == 0) {
        if (cu.item >= item_end<SK>(a)) return;
        cu = warp_bond_next_item<LT, SK>(a, warp, cu.item);
        if (cu.left == 0) return;
    }
    mbar_arrive_expect_tx(full, (fwd + L) * 16u);
    if (!cu.wrap) {
        bulk_g2s(dst, cu.src - L, (fwd + L) * 16u, full);       // [y-bonds of row y-1][rows y ..]
    } else {
        bulk_g2s(dst, cu.src + (size_t)(L - 1) * 3 * L + 2 * L, L * 16u, full);   // y-bonds of row L-1 (periodic)
        bulk_g2s(dst + L, cu.src, fwd * 16u, full);
    }
    cu.src += (size_t)3 * L * L;
    --cu.left;
}

// LT: lattice edge as a compile-time constant (shared-memory offsets become immediates), 0 = run-time a.L
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }  // conj(a) b

template <bool FIRST, int LT, int MODE, bool SK>
__global__ void __launch_bounds__(kStepThreads, 1) cheb_step_kernel(const __grid_constant__ StepArgs a)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    StepSmemHeader* hdr = reinterpret_cast<StepSmemHeader*>(smem_raw);
    double2* ring_c = reinterpret_cast<double2*>(smem_raw + kStepHeaderBytes);
    const int tid = threadIdx.x;
    const int L = LT ? LT : a.L;
    constexpr bool WP = (LT != 0);                // per-warp R_prev rings (see warp_prev_issue)
    // The per-warp rings (R_prev, bond amplitudes) are ONE stage deep, at compile time: the refill is issued the moment the warp has read
    // the stage and has a whole plane iteration to land (measured: depth 2 is not faster), and constant depths take the ring indices
    // and their wrap-around tests out of the plane loop (the J_H->inf instantiation spilled them: +3 % there).
    constexpr uint32_t kNPW = 1, kNTW = 1;
    constexpr bool TB = (MODE == kModeDex) && LT != 0 && LT <= 32;   // bond amplitudes staged through per-warp rings (see warp_bond_issue)
    constexpr int tb_units = TB ? (3 * (32 / (LT ? LT : 32)) + 1) * LT : 0;     // double2 per warp and bond stage
    double2* ring_p = ring_c + (size_t)a.nst_c * a.cstage_units;
    double2* ring_t = ring_p + (size_t)(WP ? kNPW : (uint32_t)a.nst_p) * a.pstage_units;      // per-warp bond-amplitude rings (kModeDex, compile-time L <= 32)
    // generic (slow) reduction scratch lives after the rings when requested
    double* red_slow = reinterpret_cast<double*>(ring_t + (size_t)(TB ? kNTW : 0u) * a.tstage_units);
    const bool full = LT ? (LT * LT <= kConsumerThreads) : (a.full != 0);
    const int rowu = 4 * L;                       // double2 per (y) row: 4 chunk-rows of L
    const size_t zstride = (size_t)a.P * L * rowu;  // double2 per z-plane of the whole batch

    RingCursor* cu_c = reinterpret_cast<RingCursor*>(&hdr->cur_item);
    RingCursor* cu_p = reinterpret_cast<RingCursor*>(&hdr->prev_item);
    // Programmatic dependent launch (the host sets cudaLaunchAttributeProgrammaticStreamSerialization on the step launches): this grid
    // may become resident while the previous step's grid is still draining -- one persistent CTA per SM, so a CTA of step m+1 lands on an
    // SM the moment step m's CTA there has exited.  Everything up to griddepcontrol.wait touches shared memory only (barrier init, ring
    // cursors) and overlaps the tail of step m; the wait returns once step m has COMPLETED and its writes are visible, which every
    // global access below needs (step m+1 reads the r_m that step m wrote and overwrites the r_{m-1} it read).  Both instructions are
    // no-ops in a launch without the attribute.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tid == 0) {
        for (int s = 0; s < kMaxStages; ++s) {
            mbar_init(&hdr->full_c[s], 1);
            mbar_init(&hdr->full_p[s], 1);
            mbar_init(&hdr->empty_c[s], kConsumerWarps);
            hdr->seq_c[s] = 0; hdr->rel_p[s] = 0;
        }
        cu_c->item = item_first<SK>(a); cu_c->q = -1;
        cu_p->item = item_first<SK>(a); cu_p->q = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("griddepcontrol.wait;" ::: "memory");
        // fill both rings
        for (int s = 0; s < a.nst_c; ++s) issue_cur<LT, SK>(a, cu_c, &hdr->full_c[s], ring_c + (size_t)s * a.cstage_units);
        if (!FIRST && !WP)
            for (int s = 0; s < a.nst_p; ++s) issue_prev<LT, SK>(a, cu_p, &hdr->full_p[s], ring_p + (size_t)s * a.pstage_units);
    }
    WarpPrevCursor wcu;                           // lane 0's copy is the live one
    wcu.src = nullptr; wcu.item = item_first<SK>(a) - item_stride<SK>(a); wcu.left = 0;
    WarpBondCursor tcu;                           // same for the warp's bond-amplitude ring
    tcu.src = nullptr; tcu.item = item_first<SK>(a) - item_stride<SK>(a); tcu.left = 0; tcu.wrap = 0;
    if (WP && (tid & 31) == 0) {
        // this warp's private rings: barriers, then the first planes of the warp's own sequence
        const int w = tid >> 5;
        for (int s = 0; s < kMaxWarpStages; ++s) mbar_init(&hdr->full_w[w][s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("griddepcontrol.wait;" ::: "memory");
        if (!FIRST)
            for (int s = 0; s < (int)kNPW; ++s)
                warp_prev_issue<LT, SK>(a, w, wcu, zstride, &hdr->full_w[w][s], ring_p + ((size_t)w * kNPW + s) * kWarpSegUnits);
        if (TB)
            for (int s = 0; s < (int)kNTW; ++s)
                warp_bond_issue<LT, SK>(a, w, tcu, &hdr->full_w[w][kNPW + s], ring_t + ((size_t)w * kNTW + s) * tb_units);
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");        // every thread: its own global loads (spins, bonds) and stores (r_m, Gram partials) follow
    __syncthreads();
    // R_cur stage release.  Every warp arrives on the stage's "empty" mbarrier (release semantics without a fence instruction);
    // a warp that sees the phase complete right after its own arrival refills the stage.  Two warps can see that at the same
    // time, so the refill is claimed by a relaxed CAS on the stage's refill count (== the ring pass `pass` it was consumed in).
    auto release_c = [&](uint32_t s, uint32_t pass) {
        __syncwarp();
        if ((tid & 31) == 0) {
            mbar_arrive(&hdr->empty_c[s]);
            if (mbar_test(&hdr->empty_c[s], pass & 1u) && cas_relaxed_shared(&hdr->seq_c[s], pass, pass + 1u) == pass)
                issue_cur<LT, SK>(a, cu_c, &hdr->full_c[s], ring_c + (size_t)s * a.cstage_units);
        }
    };
    auto release_p = [&](uint32_t s) {
        __syncwarp();
        if ((tid & 31) == 0 && atom_add_acq_rel_shared(&hdr->rel_p[s], 1u) == kConsumerWarps - 1) {
            hdr->rel_p[s] = 0;
            issue_prev<LT, SK>(a, cu_p, &hdr->full_p[s], ring_p + (size_t)s * a.pstage_units);
        }
    };

    // ==================================================================== consumers
    const int warp = tid >> 5, lane = tid & 31;
    // tile-local coordinates of this thread's site
    const int plane_sites = full ? L * L : a.Ty_rows * L;
    const int g = tid / plane_sites;              // pair inside the group (full mode), 0 otherwise
    const int rem = tid - g * plane_sites;
    const int yl = rem / L;
    const int x = rem - yl * L;
    const int xm = (x + L - 1) % L, xp = (x + 1) % L;

    // offset of this thread's site inside the warp's R_prev stage and the chunk stride there
    const int wp_cs = (LT != 0 && LT <= 32) ? LT : 32;
    const int wp_off = (LT != 0 && LT <= 32) ? (lane / wp_cs) * 4 * wp_cs + lane % wp_cs : lane;

    // offset of this thread's forward z bond inside the warp's bond stage: [y-bonds of row y-1][per row: z-, x-, y-bonds]
    const int tb_off = TB ? LT + (lane / (LT ? LT : 32)) * 3 * LT + lane % (LT ? LT : 32) : 0;

    uint32_t cs = 0, cpass = 0, ps = 0, pph = 0;     // next stage to consume in each ring; ring pass (R_cur) / parity (R_prev)
    uint32_t ts = 0, tph = 0;                        // bond ring: next stage, parity
    const int it_end = item_end<SK>(a), it_stride = item_stride<SK>(a);
    for (int item = item_first<SK>(a); item < it_end; item += it_stride) {
        const ItemCoord c = decode_item<SK>(a, item);
        const int p = c.pg * a.G + g;
        const bool active = (g < a.G) && (p < a.P) && (yl < c.rows);
        const int y = c.y0 + yl;

        // shared-memory offsets (double2 units, chunk 0) inside a stage
        int o_own, o_ym, o_yp, o_prev;
        if (full) {
            const int rb = g * L;
            o_own = (rb + yl) * rowu;
            o_ym = (rb + (yl + L - 1) % L) * rowu;
            o_yp = (rb + (yl + 1) % L) * rowu;
            o_prev = o_own + x;
        } else {
            o_own = (yl + 1) * rowu;
            o_ym = o_own - rowu;
            o_yp = o_own + rowu;
            o_prev = yl * rowu + x;
        }
        const int o_xm = o_own + xm, o_xp = o_own + xp;
        o_own += x; o_ym += x; o_yp += x;

        // global offset of this thread's site at plane 0 (double2 units, chunk 0)
        const size_t gsite = active ? ((size_t)p * L + y) * rowu + x : 0;
        const int site_xy = active ? (x + L * y) : 0;
        double2* outp = a.nxt + (size_t)c.z0 * zstride + gsite;    // this site's r_m at plane z (advanced per plane)

        constexpr int NG = gram_width(MODE);
        double gs[NG];                                     // Gram sums of this thread (layout: see the accumulation below)
#pragma unroll
        for (int k = 0; k < NG; ++k) gs[k] = 0.0;
        // kModeHund1: Gamma_i = (-1)^(x+y+z) of this thread's site at plane z0 (flips every plane)
        double gam = ((x + y + c.z0) & 1) ? -1.0 : 1.0;
        // kModeDex: site offsets of the -x / -y neighbours (their forward bonds are this site's backward bonds)
        const int d_xm = active ? xm - x : 0, d_ym = active ? (((y + L - 1) % L) - y) * L : 0;
        // Only the z-1 column is carried in registers; the z column is re-read from the ring stage that is resident
        // for the lateral reads anyway, the z+1 column is consumed straight into the stencil sum.
        double2 m1[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) m1[k] = make_double2(0.0, 0.0);
        // staged bonds: the backward z bond of plane z0 is the forward z bond of the site below (plane z0-1, periodic); afterwards
        // it is the forward z bond this thread read one plane earlier
        double2 tz_below = make_double2(0.0, 0.0);
        if (TB && active) tz_below = __ldg(a.Tq + ((size_t)((c.z0 + L - 1) % L) * L + y) * 3 * L + x);

        // plane z0-1: own column only
        {
            const uint32_t s = cs;
            mbar_wait(&hdr->full_c[s], cpass & 1u);
            const double2* st = ring_c + (size_t)s * a.cstage_units;
            if (active) {
#pragma unroll
                for (int k = 0; k < 4; ++k) m1[k] = st[o_own + k * L];
            }
            release_c(s, cpass);
            if (++cs == (uint32_t)a.nst_c) { cs = 0; ++cpass; }
        }
        // plane z0: stage kept for the reads of the first iteration
        uint32_t sc = cs;
        mbar_wait(&hdr->full_c[sc], cpass & 1u);
        if (++cs == (uint32_t)a.nst_c) { cs = 0; ++cpass; }

        for (int zi = 0; zi < c.nz; ++zi) {
            const int z = c.z0 + zi;
            const int si = site_xy + L * L * z;
            // spin of this site (the field is small and L2-resident); consumed after the stencil sums.  An L1 prefetch of the next
            // plane's spins (prefetch.global.L1) was measured 1.8 % SLOWER at config 4 and is not used.
            double sx = 0, sy = 0, sz = 0;
            double2 txf, txb, tyf, tyb, tzf, tzb;
            if (MODE != kModeDex) {
                sx = __ldg(a.Sx + si); sy = __ldg(a.Sy + si); sz = __ldg(a.Sz + si);
            }
            else if (!TB) {
                // bond amplitudes of this site: forward t_{i,i+e}, backward t_{i,i-e} = conj(forward bond of the neighbour)
                const int szm = site_xy + L * L * ((z + L - 1) % L);
                txf = __ldg(a.Tx + si); txb = __ldg(a.Tx + si + d_xm);
                tyf = __ldg(a.Ty + si); tyb = __ldg(a.Ty + si + d_ym);
                tzf = __ldg(a.Tz + si); tzb = __ldg(a.Tz + szm);
            }
            // plane z+1 arrives: own column
            const uint32_t sn = cs;
            mbar_wait(&hdr->full_c[sn], cpass & 1u);
            if (++cs == (uint32_t)a.nst_c) { cs = 0; ++cpass; }
            const double2* stn = ring_c + (size_t)sn * a.cstage_units;
            const double2* stc = ring_c + (size_t)sc * a.cstage_units;
            double2 acc[4], c0[4];
            if (TB && active) {                                // warp-uniform for compile-time L
                // this plane's amplitudes from the warp's bond ring
                uint64_t* bar = &hdr->full_w[warp][kNPW + ts];
                mbar_wait(bar, tph);
                const double2* stt = ring_t + ((size_t)warp * kNTW + ts) * tb_units;
                tzf = stt[tb_off]; txf = stt[tb_off + L]; txb = stt[tb_off + L + (xm - x)];
                tyf = stt[tb_off + 2 * L]; tyb = stt[tb_off - L];
                tzb = tz_below; tz_below = tzf;
            }
            if (active) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double2 p1 = stn[o_own + k * L];
                    const double2 a0 = stc[o_xm + k * L], a1 = stc[o_xp + k * L];
                    const double2 a2 = stc[o_ym + k * L], a3 = stc[o_yp + k * L];
                    c0[k] = stc[o_own + k * L];
                    if (MODE != kModeDex) {
                        acc[k] = add2(add2(add2(m1[k], p1), add2(a0, a1)), add2(a2, a3));
                    } else {
                        // sum_j t_ij x_j over the six bonds (Eq. (2)-(3))
                        acc[k] = add2(add2(add2(cmulc(tzb, m1[k]), cmul(tzf, p1)), add2(cmulc(txb, a0), cmul(txf, a1))),
                                      add2(cmulc(tyb, a2), cmul(tyf, a3)));
                    }
                }
            }
            release_c(sc, sc < cs ? cpass : cpass - 1u);       // plane z no longer needed in shared memory (sc is < nst_c behind cs)
            if (TB && active) {
                // the amplitudes are in registers (consumed by the sums above): refill the bond stage with the warp's next plane
                // (every lane orders its generic-proxy reads before the async proxy, then the warp joins, then lane 0 re-issues)
                fence_proxy_async_shared();
                __syncwarp();
                if (lane == 0)
                    warp_bond_issue<LT, SK>(a, warp, tcu, &hdr->full_w[warp][kNPW + ts], ring_t + ((size_t)warp * kNTW + ts) * tb_units);
                if (++ts == kNTW) { ts = 0; tph ^= 1; }
            }
            double2 nx[4];
            if (active) {
                if (MODE != kModeDex) {
                    const double hx = a.cj * sx, hy = a.cj * sy, hz = a.cj * sz;
#pragma unroll
                    for (int vi = 0; vi < 2; ++vi) {
                        const double2 u = c0[2 * vi], d = c0[2 * vi + 1];
                        // (h.sigma) (u,d)^T : up = hz u + (hx - i hy) d ; down = (hx + i hy) u - hz d
                        double2 hu, hd;
                        hu.x = hz * u.x + hx * d.x + hy * d.y;
                        hu.y = hz * u.y + hx * d.y - hy * d.x;
                        hd.x = hx * u.x - hy * u.y - hz * d.x;
                        hd.y = hx * u.y + hy * u.x - hz * d.y;
                        nx[2 * vi].x = a.ct * acc[2 * vi].x + hu.x;
                        nx[2 * vi].y = a.ct * acc[2 * vi].y + hu.y;
                        nx[2 * vi + 1].x = a.ct * acc[2 * vi + 1].x + hd.x;
                        nx[2 * vi + 1].y = a.ct * acc[2 * vi + 1].y + hd.y;
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < 4; ++k) { nx[k].x = a.ct * acc[k].x; nx[k].y = a.ct * acc[k].y; }
                }
            }
            if (!FIRST && WP) {
                // r_{m-2} of this site from the warp's own R_prev ring; the stage is refilled as soon as the warp has read it
                if (active) {                                  // warp-uniform for compile-time L
                    uint64_t* bar = &hdr->full_w[warp][ps];
                    mbar_wait(bar, pph);
                    double2* stp = ring_p + ((size_t)warp * kNPW + ps) * kWarpSegUnits;
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const double2 pv = stp[wp_off + k * wp_cs]; nx[k].x -= pv.x; nx[k].y -= pv.y; }
                    // The values are in registers (nx) before the refill.  Every lane orders its generic-proxy reads of the stage
                    // before the async proxy (fence.proxy.async), the warp joins, then lane 0 re-issues the bulk-TMA write into it.
                    fence_proxy_async_shared();
                    __syncwarp();
                    if (lane == 0) warp_prev_issue<LT, SK>(a, warp, wcu, zstride, bar, stp);
                    if (++ps == kNPW) { ps = 0; pph ^= 1; }
                }
            }
            if (!FIRST && !WP) {
                // r_{m-2} of this site from the R_prev ring
                const uint32_t sp = ps;
                mbar_wait(&hdr->full_p[sp], pph);
                const double2* stp = ring_p + (size_t)sp * a.pstage_units;
                if (active) {
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const double2 pv = stp[o_prev + k * L]; nx[k].x -= pv.x; nx[k].y -= pv.y; }
                }
                release_p(sp);
                if (++ps == (uint32_t)a.nst_p) { ps = 0; pph ^= 1; }
            }
            if (active) {
#pragma unroll
                for (int k = 0; k < 4; ++k) stg_stream(outp + k * L, nx[k]);
                // Gram sums <a|b> = sum conj(a) b of this site (Eq. (27)-(28)); nx = r_m, c0 = r_{m-1}
                if (MODE == kModeHund2) {
                    // vectors: up-start = chunks {0,1}, down-start = chunks {2,3}; (Yuu, Ydd, Re Yud, Im Yud, Xuu, Xdd, Re Xud, Im Xud)
                    gs[0] += nx[0].x * nx[0].x + nx[0].y * nx[0].y + nx[1].x * nx[1].x + nx[1].y * nx[1].y;
                    gs[1] += nx[2].x * nx[2].x + nx[2].y * nx[2].y + nx[3].x * nx[3].x + nx[3].y * nx[3].y;
                    gs[2] += nx[0].x * nx[2].x + nx[0].y * nx[2].y + nx[1].x * nx[3].x + nx[1].y * nx[3].y;
                    gs[3] += nx[0].x * nx[2].y - nx[0].y * nx[2].x + nx[1].x * nx[3].y - nx[1].y * nx[3].x;
                    gs[4] += c0[0].x * nx[0].x + c0[0].y * nx[0].y + c0[1].x * nx[1].x + c0[1].y * nx[1].y;
                    gs[5] += c0[2].x * nx[2].x + c0[2].y * nx[2].y + c0[3].x * nx[3].x + c0[3].y * nx[3].y;
                    gs[6] += c0[0].x * nx[2].x + c0[0].y * nx[2].y + c0[1].x * nx[3].x + c0[1].y * nx[3].y;
                    gs[7] += c0[0].x * nx[2].y - c0[0].y * nx[2].x + c0[1].x * nx[3].y - c0[1].y * nx[3].x;
                } else if (MODE == kModeHund1) {
                    // per site q of the slot, from the up-start vector (u, d) = nx, (u', d') = c0 alone:
                    //   Y = <r_m|r_m>, X = Re <r_{m-1}|r_m>, W = sum_i Gamma_i (u'_i d_i - d'_i u_i)
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        const double2 u = nx[2 * q], d = nx[2 * q + 1], up = c0[2 * q], dp = c0[2 * q + 1];
                        gs[4 * q + 0] += u.x * u.x + u.y * u.y + d.x * d.x + d.y * d.y;
                        gs[4 * q + 1] += up.x * u.x + up.y * u.y + dp.x * d.x + dp.y * d.y;
                        gs[4 * q + 2] += gam * (up.x * d.x - up.y * d.y - dp.x * u.x + dp.y * u.y);
                        gs[4 * q + 3] += gam * (up.x * d.y + up.y * d.x - dp.x * u.y - dp.y * u.x);
                    }
                } else {
                    // per site q of the slot, start vectors o = chunk 2q, v = chunk 2q+1:
                    //   (Yoo, Yvv, Re Yov, Im Yov, Xoo, Xvv, Re Xov, Im Xov), X(a,b) = <r^a_{m-1}|r^b_m>
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
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) m1[k] = c0[k];
            }
            outp += zstride;
            gam = -gam;
            sc = sn;
        }
        // the upper halo plane (z0+nz) was only needed for the own column
        release_c(sc, sc < cs ? cpass : cpass - 1u);

        // ---------------------------------------------------------- per-item reduction of the 8 Gram sums
        const int ntiles = SK ? a.ntiles : a.nty * a.nzc;
        const int tile = SK ? c.zc : c.ty * a.nzc + c.zc;
        const int npairs_cta = full ? a.G : 1;
        if (!a.slow_reduce) {
            // every warp lies inside one slot: shuffle, then combine the warps of each slot in fixed order
#pragma unroll
            for (int k = 0; k < NG; ++k) {
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) gs[k] += __shfl_xor_sync(0xffffffffu, gs[k], off);
            }
            if (lane == 0) {
#pragma unroll
                for (int k = 0; k < NG; ++k) hdr->red[warp * 16 + k] = gs[k];
            }
            consumer_bar_sync();
            const int wpp = plane_sites / 32;                  // warps per slot
            for (int idx = tid; idx < NG * npairs_cta; idx += kConsumerThreads) {
                const int gg = idx / NG, k = idx % NG;
                const int pp = c.pg * a.G + gg;
                if (pp < a.P) {
                    double sacc = 0.0;
                    for (int w = gg * wpp; w < (gg + 1) * wpp; ++w) sacc += hdr->red[w * 16 + k];
                    a.gram[((size_t)pp * ntiles + tile) * NG + k] = sacc;
                }
            }
            consumer_bar_sync();
        } else {
#pragma unroll
            for (int k = 0; k < NG; ++k) red_slow[tid * NG + k] = gs[k];
            consumer_bar_sync();
            for (int idx = tid; idx < NG * npairs_cta; idx += kConsumerThreads) {
                const int gg = idx / NG, k = idx % NG;
                const int pp = c.pg * a.G + gg;
                if (pp < a.P) {
                    double sacc = 0.0;
                    for (int t2 = gg * plane_sites; t2 < (gg + 1) * plane_sites; ++t2) sacc += red_slow[t2 * NG + k];
                    a.gram[((size_t)pp * ntiles + tile) * NG + k] = sacc;
                }
            }
            consumer_bar_sync();
        }
    }
}

}  // namespace gfmc
