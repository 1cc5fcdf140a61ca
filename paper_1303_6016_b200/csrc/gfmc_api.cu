// gfmc_api.cu -- C ABI of libgfmc.so (include/gfmc.h): context, workspace, host orchestration.
// Every step of the hot path runs in the kernels of cheb_step.cuh / post.cuh; the host code below only
// validates, sizes, schedules launches and moves user buffers.  There is no CPU fallback.
#include "../../include/gfmc.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>     // header-only NVTX v3: ranges around every public call (visible in nsys / ncu timelines; no link dependency)

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "cheb_step.cuh"
#include "cheb_resident.cuh"
#include "post.cuh"
#include "exact_batch.cuh"
#include "cheb_step2.cuh"

using namespace gfmc;

namespace {

thread_local std::string g_create_error;

struct StepPlan {
    int full, G, Ty, nty, nzc, nzper, npg, nitems, nst_c, nst_p, nst_t, cstage_units, pstage_units, tstage_units, slow_reduce, grid;
    size_t smem_bytes;
    int ntiles;       // nty * nzc : Gram partials per pair per step
    bool pdl;         // step launches use programmatic dependent launch (default; GFMC_FLAG_NO_PDL turns it off)
    bool ok;
};

// lattice edges with a compile-time instantiation of the step kernel; every other L runs the generic one
#define GFMC_FOR_EACH_LT_SPECIFIC(X) X(8) X(16) X(32) X(64)
#define GFMC_FOR_EACH_LT(X) X(0) GFMC_FOR_EACH_LT_SPECIFIC(X)

bool has_compile_time_L(int L)
{
#define X(LT_) if (L == LT_) return true;
    GFMC_FOR_EACH_LT_SPECIFIC(X)
#undef X
    return false;
}

// Diagnostic overrides of one context (gfmc_params.flags / ring_stages_* / streamk_eff).  Nothing here is process-wide: two
// contexts with different settings can live side by side and creating one never changes another.
struct Tuning {
    int nst_c = 0, nst_p = 0;             // ring depths of the streaming kernel, 0 = automatic
    bool no_resident = false;             // small lattices also run the streaming kernel (A/B measurements)
    bool green_direct = false;            // Green's functions by the direct O(M K) sum even where the FFT kernel applies
    bool no_graph = false;                // sweeps launch every kernel individually (no CUDA graph replay)
    bool no_pdl = false;                  // step launches without programmatic dependent launch (A/B measurements)
    bool two_step = false;                // one-vector mode at L = 32: two Chebyshev steps per pass (cheb_step2.cuh)
    double streamk_eff = 0.97;            // use the explicit work list when the arithmetic one wastes more than this (<= 0: never)
};
Tuning tuning_of(const gfmc_params* p)
{
    Tuning t;
    t.nst_c = p->ring_stages_cur; t.nst_p = p->ring_stages_prev;
    t.no_resident = (p->flags & GFMC_FLAG_NO_RESIDENT) != 0;
    t.green_direct = (p->flags & GFMC_FLAG_GREEN_DIRECT) != 0;
    t.no_graph = (p->flags & GFMC_FLAG_NO_GRAPH) != 0;
    t.no_pdl = (p->flags & GFMC_FLAG_NO_PDL) != 0;
    t.two_step = (p->flags & GFMC_FLAG_TWO_STEP) != 0;
    t.streamk_eff = p->streamk_eff == 0.0 ? 0.97 : p->streamk_eff;
    return t;
}

// Work decomposition of one fused step for P pairs ("tiling").
StepPlan make_plan(int L, int P, int nSM, size_t smem_limit, int NG, const Tuning& tun)
{
    StepPlan pl{};
    const int plane = L * L;
    int rows;
    if (plane <= kConsumerThreads) {
        pl.full = 1; pl.Ty = L; pl.nty = 1;
        int G = std::min(64, kConsumerThreads / plane);
        while (G > 1 && (P + G - 1) / G < nSM) G = (G + 1) / 2;      // keep at least one item per SM if possible
        pl.G = G;
        rows = G * L;
    } else {
        pl.full = 0; pl.G = 1;
        const int tymax = std::max(1, kConsumerThreads / L);
        pl.nty = (L + tymax - 1) / tymax;
        pl.Ty = (L + pl.nty - 1) / pl.nty;
        pl.nty = (L + pl.Ty - 1) / pl.Ty;
        rows = pl.Ty + 2;
    }
    pl.npg = (P + pl.G - 1) / pl.G;
    const int base_items = pl.npg * pl.nty;
    int nzc = 1;
    if (base_items < nSM) nzc = std::min(std::max(1, L / 4), (nSM + base_items - 1) / base_items);
    pl.nzper = (L + nzc - 1) / nzc;
    pl.nzc = (L + pl.nzper - 1) / pl.nzper;
    pl.nitems = base_items * pl.nzc;
    pl.ntiles = pl.nty * pl.nzc;
    pl.cstage_units = rows * 4 * L;
    pl.pstage_units = (pl.full ? rows : pl.Ty) * 4 * L;
    // compile-time lattice edges stream R_prev through per-warp rings: 16 warps x 2 KiB per stage whatever G is
    const bool warp_prev = has_compile_time_L(L);
    if (warp_prev) pl.pstage_units = kConsumerWarps * kWarpSegUnits;
    // J_H->inf model (NG = 16) with compile-time L <= 32: the bond amplitudes stream through per-warp rings as well
    const bool bond_rings = (NG == 16) && warp_prev && L <= 32;
    pl.tstage_units = bond_rings ? kConsumerWarps * (3 * (32 / L) + 1) * L : 0;
    pl.nst_t = bond_rings ? 1 : 0;
    const int np_max = warp_prev ? (bond_rings ? kMaxWarpStages - 2 : kMaxWarpStages) : kMaxStages;
    const size_t cbytes = (size_t)pl.cstage_units * 16, pbytes = (size_t)pl.pstage_units * 16, tbytes = (size_t)pl.tstage_units * 16;
    const int plane_sites = pl.full ? plane : pl.Ty * L;
    pl.slow_reduce = (plane_sites % 32 != 0) ? 1 : 0;
    const size_t extra = pl.slow_reduce ? (size_t)kConsumerThreads * NG * sizeof(double) : 0;
    if (smem_limit < kStepHeaderBytes + extra + 3 * cbytes + pbytes + tbytes || L > kConsumerThreads) { pl.ok = false; return pl; }
    // ring depths: as deep as shared memory allows, R_cur ring one stage deeper than the R_prev ring
    // (the consumers hold two R_cur planes but only one R_prev slab)
    const size_t budget = smem_limit - kStepHeaderBytes - extra - tbytes;
    int nc = 3, np = 1;
    for (;;) {
        if (nc < kMaxStages && nc <= np + 1 && (nc + 1) * cbytes + np * pbytes <= budget) { ++nc; continue; }
        if (np < np_max && (size_t)nc * cbytes + (np + 1) * pbytes <= budget) { ++np; continue; }
        if (nc < kMaxStages && (nc + 1) * cbytes + np * pbytes <= budget) { ++nc; continue; }
        break;
    }
    // Measured (round 2, same-box A/B at configs 3, 4, 5, sustained step loops): for the Eq. (1) modes with per-warp R_prev rings the SHALLOWEST
    // legal rings are the fastest -- (3, 1) against the deepest that fit, (4, 2): +1.2 % at config 4, +2.9 % at config 3, +1.9 % at config 5
    // (one plane of R_cur in flight beside the two being read is enough to cover HBM latency at 2.3 us per plane; more prefetch only adds
    // shared-memory and L2 traffic under the power cap).  The J_H->inf mode keeps (4, 1, 1): 1.278 against 1.289 ms with (3, 1).
    if (warp_prev && !bond_rings) nc = 3;
    if (tun.nst_c > 0) nc = tun.nst_c;
    if (tun.nst_p > 0) np = std::min(tun.nst_p, np_max);
    if (warp_prev) np = 1;               // the per-warp rings are one stage deep at compile time (cheb_step.cuh); ring_stages_prev applies to run-time L only
    pl.nst_c = nc; pl.nst_p = np;
    pl.smem_bytes = kStepHeaderBytes + (size_t)nc * cbytes + (size_t)np * pbytes + (size_t)pl.nst_t * tbytes + extra;
    if (pl.smem_bytes > smem_limit || nc < 3 || np < 1) { pl.ok = false; return pl; }
    pl.grid = std::min(pl.nitems, nSM);
    // only launches that fill the machine: a grid smaller than the SM count would let the NEXT launches become resident on the free SMs at once and
    // sit there waiting, taking those SMs away from other streams (concurrent chains of small batches)
    pl.pdl = !tun.no_pdl && pl.grid >= nSM;
    pl.ok = true;
    return pl;
}

// One step launch.  With pdl the launch carries cudaLaunchAttributeProgrammaticStreamSerialization: the grid may start while the previous
// kernel of the stream drains, and waits inside the kernel (griddepcontrol.wait, cheb_step.cuh) before its first global access.
template <class Kernel>
void launch_step_kernel(Kernel kernel, const StepPlan& pl, const StepArgs& sa, cudaStream_t st)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)pl.grid); cfg.blockDim = dim3(kStepThreads); cfg.dynamicSmemBytes = pl.smem_bytes; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pl.pdl ? 1 : 0;
    (void)cudaLaunchKernelEx(&cfg, kernel, sa);            // errors surface through cudaGetLastError at the call sites, as with <<<>>>
}

template <int MODE>
void launch_step_mode(int L, bool first, const StepPlan& pl, const StepArgs& sa, cudaStream_t st)
{
#define X(LT_)                                                                                                \
    if (L == LT_ || LT_ == 0) {                                                                               \
        if (sa.items) {                                                                                       \
            if (first) launch_step_kernel(cheb_step_kernel<true, LT_, MODE, true>, pl, sa, st);               \
            else       launch_step_kernel(cheb_step_kernel<false, LT_, MODE, true>, pl, sa, st);              \
        } else {                                                                                              \
            if (first) launch_step_kernel(cheb_step_kernel<true, LT_, MODE, false>, pl, sa, st);              \
            else       launch_step_kernel(cheb_step_kernel<false, LT_, MODE, false>, pl, sa, st);             \
        }                                                                                                     \
        return;                                                                                               \
    }
    GFMC_FOR_EACH_LT_SPECIFIC(X)
    X(0)
#undef X
}

void launch_step(int mode, int L, bool first, const StepPlan& pl, const StepArgs& sa, cudaStream_t st)
{
    if (mode == kModeHund2) launch_step_mode<kModeHund2>(L, first, pl, sa, st);
    else if (mode == kModeHund1) launch_step_mode<kModeHund1>(L, first, pl, sa, st);
    else launch_step_mode<kModeDex>(L, first, pl, sa, st);
}

template <int MODE>
cudaError_t set_step_smem_limit_mode(int bytes)
{
    cudaError_t e = cudaSuccess;
#define X(LT_)                                                                                                          \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_step_kernel<true, LT_, MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);  \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_step_kernel<false, LT_, MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes); \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_step_kernel<true, LT_, MODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);   \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_step_kernel<false, LT_, MODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    GFMC_FOR_EACH_LT(X)
#undef X
    return e;
}

cudaError_t set_step_smem_limit(int bytes)
{
    cudaError_t e = set_step_smem_limit_mode<kModeHund2>(bytes);
    if (e == cudaSuccess) e = set_step_smem_limit_mode<kModeHund1>(bytes);
    if (e == cudaSuccess) e = set_step_smem_limit_mode<kModeDex>(bytes);
    return e;
}

// Small lattices (L^3 <= 512 sites, Eq. (1) modes): both work vectors of a slot live in shared memory for the whole recursion
// (cheb_resident.cuh).  G slots per CTA, each padded to whole warps.
struct ResidentPlan { bool ok; int Npad, G, spt; size_t smem_bytes; };
constexpr int kResMaxSpt = 4;             // sites per thread: L^3 <= 4 * 512 and 128 L^3 bytes of shared memory, i.e. L <= 12
ResidentPlan make_resident_plan(int L, size_t smem_limit, const Tuning& tun)
{
    ResidentPlan rp{};
    const long long N = (long long)L * L * L;
    if (tun.no_resident || N > (long long)kResMaxSpt * kResThreads) return rp;
    if (N <= kResThreads) {
        rp.spt = 1;
        rp.Npad = (int)((N + 31) / 32 * 32);
        rp.G = kResThreads / rp.Npad;
    } else {
        rp.spt = (int)((N + kResThreads - 1) / kResThreads);
        rp.Npad = kResThreads;
        rp.G = 1;
    }
    rp.smem_bytes = resident_smem_bytes((int)N, rp.G);
    rp.ok = rp.G >= 1 && rp.smem_bytes <= smem_limit;
    return rp;
}

template <int MODE>
void launch_resident_mode(int spt, unsigned grid, size_t smem, cudaStream_t st, const ResidentArgs& ra)
{
    if (spt == 1) cheb_resident_kernel<MODE, 1><<<grid, kResThreads, smem, st>>>(ra);
    else if (spt == 2) cheb_resident_kernel<MODE, 2><<<grid, kResThreads, smem, st>>>(ra);
    else if (spt == 3) cheb_resident_kernel<MODE, 3><<<grid, kResThreads, smem, st>>>(ra);
    else cheb_resident_kernel<MODE, 4><<<grid, kResThreads, smem, st>>>(ra);
}

template <int MODE>
cudaError_t set_resident_smem_limit_mode(int bytes)
{
    cudaError_t e = cudaFuncSetAttribute(cheb_resident_kernel<MODE, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_resident_kernel<MODE, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_resident_kernel<MODE, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_resident_kernel<MODE, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    return e;
}

// mode of the fused step for a parameter set, and the number of 4-chunk slots P sites occupy in the work buffers
int mode_of(const gfmc_params* p) { return p->model == GFMC_MODEL_DEX_INF ? kModeDex : (p->ph_symmetry ? kModeHund1 : kModeHund2); }
int slots_of(int mode, int P) { return mode == kModeHund2 ? P : (P + 1) / 2; }

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

struct Layout {            // byte offsets into the arena
    size_t R2, R3;             // two-steps-per-pass mode: the pass cannot run in place, four work buffers
    size_t xmu, xG;            // exact batches: cross moments [Pe][Pe][M][4], Green blocks [Pe][Pe][K][4] (complex)
    size_t R0, R1, Sx, Sy, Sz, Saos, Tx, Ty, Tz, Tq, vnorm2, gram, mu, tw, w, sites, order, prop, uni, dS, acc, Gbuf, scal, logdS, logacc, items, cta_start, total;
    size_t max_items;
    size_t gram_doubles_per_step;
    int g_chunk;
};

bool valid_params(const gfmc_params* p)
{
    if (!p) return false;
    if (p->L < 2 || p->L > 256) return false;
    if (p->model != GFMC_MODEL_HUND && p->model != GFMC_MODEL_DEX_INF) return false;
    if (p->model == GFMC_MODEL_DEX_INF && (p->L < 3 || p->ph_symmetry)) return false;
    if (p->ph_symmetry != 0 && p->ph_symmetry != 1) return false;
    if (p->ph_symmetry && (p->L & 1)) return false;            // the shortcut needs a bipartite (even-L) periodic lattice
    if (p->M < 2 || (p->M & 1)) return false;
    if (p->n_energy < 0) return false;
    if (!(p->T > 0.0) || !std::isfinite(p->T) || !std::isfinite(p->t) || !std::isfinite(p->JH) || !std::isfinite(p->mu)) return false;
    if (p->kernel < 0 || p->kernel > 2) return false;
    if (p->max_batch_sites < 1) return false;
    if (p->flags & ~(GFMC_FLAG_NO_RESIDENT | GFMC_FLAG_GREEN_DIRECT | GFMC_FLAG_NO_GRAPH | GFMC_FLAG_TWO_STEP | GFMC_FLAG_NO_PDL)) return false;
    // two steps per pass: built for the one-vector mode on the 32^3 lattice, an even number of fused steps
    if ((p->flags & GFMC_FLAG_TWO_STEP) && !(p->model == GFMC_MODEL_HUND && p->ph_symmetry && p->L == k2L && p->M % 4 == 0)) return false;
    if (p->ring_stages_cur != 0 && (p->ring_stages_cur < 3 || p->ring_stages_cur > kMaxStages)) return false;
    if (p->ring_stages_prev != 0 && (p->ring_stages_prev < 1 || p->ring_stages_prev > kMaxStages)) return false;
    if (!std::isfinite(p->streamk_eff) || p->streamk_eff > 1.0) return false;
    // exactness inside a batch (f5): Eq. (1) with both start vectors only (the flip is an on-site 2x2 block), small batches
    if (p->exact_batch_sites < 0 || p->exact_batch_sites > 64 || p->exact_batch_sites > p->max_batch_sites) return false;
    if (p->exact_batch_sites > 0 && (p->model != GFMC_MODEL_HUND || p->ph_symmetry)) return false;
    if (p->model == GFMC_MODEL_HUND && 6.0 * std::fabs(p->t) + std::sqrt(2.0) * std::fabs(p->JH) <= 0.0) return false;
    if (p->model == GFMC_MODEL_DEX_INF && !(std::fabs(p->t) > 0.0)) return false;
    return true;
}

// nSM / smem_limit are device properties; for sizing without a device the B200 values are assumed.
Layout make_layout(const gfmc_params* p, int nSM, size_t smem_limit)
{
    Layout l{};
    const size_t N = (size_t)p->L * p->L * p->L;
    const size_t B = (size_t)p->max_batch_sites;
    const size_t M = (size_t)p->M;
    const size_t K = p->n_energy > 0 ? (size_t)p->n_energy : 2 * M;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    const int mode = mode_of(p);
    const int NG = gram_width(mode);
    const Tuning tun = tuning_of(p);
    const size_t Bs = (size_t)slots_of(mode, (int)B);       // 4-chunk slots: B (two vectors x two spin components per site) or ceil(B/2)
    const size_t rbytes = 64 * N * Bs;                      // 16 B * N sites * 4 chunks * slots
    l.R0 = take(rbytes); l.R1 = take(rbytes);
    l.R2 = take(tun.two_step ? rbytes : 0); l.R3 = take(tun.two_step ? rbytes : 0);
    l.Sx = take(8 * N); l.Sy = take(8 * N); l.Sz = take(8 * N); l.Saos = take(24 * N);
    l.Tx = take(16 * N); l.Ty = take(16 * N); l.Tz = take(16 * N); l.Tq = take(48 * N); l.vnorm2 = take(8 * B);
    // Gram partials per step: P * ntiles * 8 doubles.  ntiles > nty only while P is too small to fill the SMs,
    // so the maximum over P <= B is reached either at such a small P or at P = B.
    size_t gmax = 0;
    const size_t small = std::min<size_t>(Bs, (size_t)nSM * 64 + 1);
    for (size_t P = 1; P <= small; ++P)
        gmax = std::max(gmax, P * (size_t)make_plan(p->L, (int)P, nSM, smem_limit, NG, tun).ntiles * NG);
    const StepPlan plB = make_plan(p->L, (int)Bs, nSM, smem_limit, NG, tun);
    gmax = std::max(gmax, Bs * (size_t)plB.ntiles * NG);
    gmax = std::max(gmax, Bs * (size_t)2 * plB.nty * NG);      // explicit work list: up to two z pieces per (pair group, y-tile) column
    l.gram_doubles_per_step = gmax;
    l.gram = take(gmax * 8 * (M / 2));
    l.mu = take(B * M * 4 * 16);
    l.tw = take(4 * K * 16);
    l.w = take(M * 8);
    l.sites = take(B * 4); l.order = take(N * 4);
    l.prop = take(std::max(B, N) * 24); l.uni = take(std::max(B, N) * 8);
    l.dS = take(B * 8); l.acc = take(B);
    l.g_chunk = (int)std::min<size_t>(B, std::max<size_t>(1, ((size_t)64 << 20) / (K * 64)));
    l.Gbuf = take((size_t)l.g_chunk * K * 64);
    l.scal = take(256);
    const size_t Pe = (size_t)p->exact_batch_sites;
    l.xmu = take(Pe * Pe * M * 64); l.xG = take(Pe * Pe * K * 64);
    l.logdS = take(N * 8); l.logacc = take(N);
    l.max_items = Bs * (size_t)std::max(1, plB.nty) + (size_t)nSM + 16;
    // two explicit work lists side by side (a sweep alternates between a full and a short last batch)
    l.items = take(2 * l.max_items * sizeof(WorkItem)); l.cta_start = take(2 * ((size_t)nSM + 2) * 4);
    l.total = off;
    return l;
}

}  // namespace

struct gfmc_ctx {
    gfmc_params p;
    int N, D, K;
    int mode;                            // kModeHund2 / kModeHund1 / kModeDex
    double a, b, lambda;
    cudaStream_t stream;
    int nSM;
    size_t smem_limit;
    char* arena;
    bool own_arena;
    Layout lay;
    bool spins_set;
    std::string err;
    int64_t counts[2];
    std::vector<int32_t> order_h;       // colour-major site order
    int ncolour[2];
    Tuning tun;                          // per-context diagnostic overrides (gfmc_params.flags, ...)
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev_pool;   // at most kMaxTimedBatches pairs: later batches of a call are not timed
    size_t ev_used;
    int64_t loop_steps, loop_vectors;
    double loop_ms;
    void* pinned;                        // small pinned staging buffer
    size_t pinned_bytes;
    // CUDA graphs of one frozen-batch update inside a sweep (launch-bound regime), keyed by everything that is baked into the nodes
    struct BatchGraph { int P; const double* prop; const double* uni; double* dlog; uint8_t* alog; double T; cudaGraphExec_t exec; int64_t n0, n1; uint64_t used; };
    std::vector<BatchGraph> graphs;      // small LRU cache
    uint64_t graph_clock;
    bool capturing;
    struct WorkList { int slots, ntiles; uint64_t used; } sk[2];   // explicit work lists on the device: built for this many slots (0 = none)
    uint64_t sk_clock;
    bool own_stream;                     // params.stream was NULL: the context runs on its own stream, ordered after the legacy stream per call
    cudaEvent_t legacy_ev;
    cudaEvent_t throttle_ev[2];          // bound the host's run-ahead in long sweeps (see sweep_device)
    long throttle_n;
    int batch_mode;                      // GFMC_BATCH_FROZEN / GFMC_BATCH_EXACT: how gfmc_update_batch / gfmc_sweep / gfmc_run decide inside a batch
    int64_t run_sweeps;                  // sweeps of the most recent gfmc_run (its running statistics live on the device, scal[24..27])

    template <class T> T* ptr(size_t off) const { return reinterpret_cast<T*>(arena + off); }
};

namespace {

int fail(gfmc_ctx* c, int code, const char* fmt, ...)
{
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
    if (c) c->err = buf; else g_create_error = buf;
    return code;
}

#define CU_TRY(ctx, expr)                                                                           \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return fail(ctx, GFMC_ECUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

int copy_in(gfmc_ctx* c, void* dst_dev, const void* src, size_t bytes, int mem)
{
    CU_TRY(c, cudaMemcpyAsync(dst_dev, src, bytes, mem == GFMC_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, c->stream));
    return GFMC_OK;
}
int copy_out(gfmc_ctx* c, void* dst, const void* src_dev, size_t bytes, int mem)
{
    CU_TRY(c, cudaMemcpyAsync(dst, src_dev, bytes, mem == GFMC_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->stream));
    return GFMC_OK;
}

void begin_call(gfmc_ctx* c)
{
    c->ev_used = 0; c->loop_steps = 0; c->loop_vectors = 0; c->loop_ms = 0.0; c->err.clear();
    if (c->own_stream) {
        // the caller asked for "the default stream": everything queued on the legacy stream so far precedes this call
        // (every call ends with a synchronisation of the context's stream, so later legacy-stream work follows it)
        cudaSetDevice(c->p.device);
        if (cudaEventRecord(c->legacy_ev, cudaStreamLegacy) == cudaSuccess) cudaStreamWaitEvent(c->stream, c->legacy_ev, 0);
    }
}

int end_call(gfmc_ctx* c)
{
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    double ms = 0.0;
    for (size_t i = 0; i < c->ev_used; ++i) {
        float t = 0.f;
        CU_TRY(c, cudaEventElapsedTime(&t, c->ev_pool[i].first, c->ev_pool[i].second));
        ms += t;
    }
    c->loop_ms = ms;
    return GFMC_OK;
}

// Every public entry point that queues work holds one of these.  Whatever path the call leaves by -- including every error
// return -- the context's stream has drained before the API returns, so caller buffers are no longer in use and the header's
// "synchronous on return" holds; finish() additionally collects the step-loop timing.  The first error code is the one returned.
struct CallGuard {
    gfmc_ctx* c; bool done = false;
    CallGuard(gfmc_ctx* c_, const char* name) : c(c_) { nvtxRangePushA(name); begin_call(c); }
    int finish() { done = true; return end_call(c); }
    ~CallGuard()
    {
        if (!done) { std::string keep = c->err; cudaStreamSynchronize(c->stream); (void)cudaGetLastError(); c->err = keep; }
        nvtxRangePop();
    }
    CallGuard(const CallGuard&) = delete; CallGuard& operator=(const CallGuard&) = delete;
};

// Step-loop timing: at most kMaxTimedBatches event pairs per call (a sequential sweep on a large lattice has thousands of batches;
// timing the first ones is enough for an average and keeps the event pool bounded).  Returns nullptr when this batch is not timed.
constexpr size_t kMaxTimedBatches = 64;
std::pair<cudaEvent_t, cudaEvent_t>* next_timing_events(gfmc_ctx* c)
{
    if (c->capturing || c->ev_used >= kMaxTimedBatches) return nullptr;
    if (c->ev_used == c->ev_pool.size()) {
        cudaEvent_t e0, e1;
        if (cudaEventCreate(&e0) != cudaSuccess) return nullptr;
        if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return nullptr; }
        c->ev_pool.emplace_back(e0, e1);
    }
    return &c->ev_pool[c->ev_used++];
}

// forward bond amplitudes of Eq. (3) from the current spins (kModeDex only)
int refresh_bonds(gfmc_ctx* c)
{
    if (c->mode != kModeDex) return GFMC_OK;
    dex_bonds_kernel<<<(c->N + 127) / 128, 128, 0, c->stream>>>(c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy), c->ptr<double>(c->lay.Sz),
                                                               c->ptr<double2>(c->lay.Tx), c->ptr<double2>(c->lay.Ty), c->ptr<double2>(c->lay.Tz),
                                                               c->ptr<double2>(c->lay.Tq), c->p.L);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return GFMC_OK;
}

// Explicit work list of the streaming kernel ("stream-K" decomposition).  The arithmetic enumeration hands out whole (pair group,
// y-tile) columns of L planes, so a launch takes ceil(columns / CTAs) rounds: 1.73 rounds of work cost 2 at config 3.  Here the
// columns x planes are cut into one contiguous range per CTA instead (boundaries snapped so that no piece is shorter than 2 planes);
// a column that straddles two CTAs becomes two z pieces, each re-reading its two halo planes.  Used when every CTA gets at least
// two columns (so a column is cut at most once: two Gram tiles per y-tile) and the arithmetic enumeration wastes more than
// 1 - streamk_eff of a launch.  Returns false if not applicable.
bool streamk_applicable(const StepPlan& pl, int L, int nSM, double streamk_eff)
{
    if (streamk_eff <= 0.0 || pl.nzc != 1 || L < 4) return false;
    const long long C = (long long)pl.npg * pl.nty;
    if (C * L < (long long)nSM * (L + 4)) return false;      // every CTA's range exceeds a column by 4 planes: at most one cut per column
    const double eff = (double)C / (double)(((C + nSM - 1) / nSM) * nSM);
    return eff < streamk_eff;
}
// Returns (in *which) the index of the device-side list built for Ps slots; two lists are cached (LRU) because a sweep alternates
// between the full batch size and a short last batch.
int upload_item_table(gfmc_ctx* c, const StepPlan& pl, int Ps, int* which)
{
    for (int k = 0; k < 2; ++k)
        if (c->sk[k].slots == Ps) { c->sk[k].used = ++c->sk_clock; *which = k; return GFMC_OK; }
    const int slot = (c->sk[0].slots == 0 || (c->sk[1].slots != 0 && c->sk[0].used < c->sk[1].used)) ? 0 : 1;
    *which = slot;
    const int L = c->p.L, grid = c->nSM;
    const long long C = (long long)pl.npg * pl.nty, U = C * L;
    std::vector<WorkItem> items;
    std::vector<int> start(grid + 1, 0);
    items.reserve((size_t)C + grid);
    auto bound = [&](int b) {
        long long u = (U * b + grid / 2) / grid;
        const long long r = u % L;
        if (r < 2) u -= r; else if (L - r < 2) u += L - r;
        return std::min(u, U);
    };
    for (int b = 0; b < grid; ++b) {
        start[b] = (int)items.size();
        long long u = bound(b);
        const long long e = (b + 1 == grid) ? U : bound(b + 1);
        while (u < e) {
            const long long col = u / L;
            const int z0 = (int)(u % L);
            const int nz = (int)std::min<long long>(L - z0, e - u);
            items.push_back(WorkItem{(int)(col / pl.nty), (int)(col % pl.nty), z0, nz, (int)(col % pl.nty) * 2 + (z0 > 0 ? 1 : 0)});
            u += nz;
        }
    }
    start[grid] = (int)items.size();
    if (items.size() > c->lay.max_items) return fail(c, GFMC_ENOMEM, "work list too long");
    c->sk[slot].slots = 0;
    CU_TRY(c, cudaMemcpyAsync(c->ptr<WorkItem>(c->lay.items) + (size_t)slot * c->lay.max_items, items.data(), items.size() * sizeof(WorkItem),
                              cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaMemcpyAsync(c->ptr<int>(c->lay.cta_start) + (size_t)slot * (c->nSM + 2), start.data(), start.size() * sizeof(int),
                              cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));        // the host vectors die here
    c->sk[slot].slots = Ps; c->sk[slot].ntiles = 2 * pl.nty; c->sk[slot].used = ++c->sk_clock;
    return GFMC_OK;
}

// a2 + a3 + moment read-out with the vectors resident in shared memory (L^3 <= 512): ONE launch runs all M/2 steps.
int run_moments_resident(gfmc_ctx* c, int P, int Ps, const ResidentPlan& rp, const double* prop_dev, int by_site)
{
    const int M = c->p.M, mode = c->mode;
    const int NG = gram_width(mode);
    if ((size_t)Ps * NG > c->lay.gram_doubles_per_step) return fail(c, GFMC_ENOMEM, "gram scratch too small");
    auto* ev = next_timing_events(c);             // the step-loop events are not recorded into a CUDA graph
    ResidentArgs ra{};
    ra.sites = c->ptr<int32_t>(c->lay.sites);
    if (mode == kModeDex) {
        // |o>, |v> = Delta|o> (Eq. (21)) and <v|v> by the same kernel as the streaming path, into the (small) global buffer R0;
        // the resident kernel copies its slots from there
        double2* R0 = c->ptr<double2>(c->lay.R0);
        CU_TRY(c, cudaMemsetAsync(R0, 0, (size_t)64 * c->N * Ps, c->stream));
        init_start_vectors_dex<<<(P + 127) / 128, 128, 0, c->stream>>>(R0, ra.sites, prop_dev, by_site, c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy),
                                                                       c->ptr<double>(c->lay.Sz), c->p.t, c->ptr<double>(c->lay.vnorm2), P, Ps, c->p.L);
        c->counts[1] += 1;
        ra.R0 = R0;
        ra.Tx = c->ptr<double2>(c->lay.Tx); ra.Ty = c->ptr<double2>(c->lay.Ty); ra.Tz = c->ptr<double2>(c->lay.Tz);
    }
    if (ev) CU_TRY(c, cudaEventRecord(ev->first, c->stream));
    ra.Sx = c->ptr<double>(c->lay.Sx); ra.Sy = c->ptr<double>(c->lay.Sy); ra.Sz = c->ptr<double>(c->lay.Sz);
    ra.gram = c->ptr<double>(c->lay.gram);
    ra.t_over_a = c->p.t / c->a; ra.jh_over_a = (mode == kModeDex) ? 0.0 : c->p.JH / c->a;
    ra.L = c->p.L; ra.N = c->N; ra.Npad = rp.Npad; ra.G = rp.G; ra.P = P; ra.Ps = Ps; ra.nsteps = M / 2;
    const unsigned grid = (unsigned)((Ps + rp.G - 1) / rp.G);
    if (mode == kModeHund2) launch_resident_mode<kModeHund2>(rp.spt, grid, rp.smem_bytes, c->stream, ra);
    else if (mode == kModeHund1) launch_resident_mode<kModeHund1>(rp.spt, grid, rp.smem_bytes, c->stream, ra);
    else launch_resident_mode<kModeDex>(rp.spt, grid, rp.smem_bytes, c->stream, ra);
    c->counts[0] += 1;
    if (ev) c->loop_steps += M / 2;
    c->loop_vectors = (mode == kModeHund1) ? (int64_t)P : 2 * (int64_t)P;
    if (ev) CU_TRY(c, cudaEventRecord(ev->second, c->stream));
    const long long nthreads = (long long)P * (M / 2 + 1);
    const unsigned nblk = (unsigned)((nthreads + 255) / 256);
    double2* mu = c->ptr<double2>(c->lay.mu);
    if (mode == kModeHund2) finalize_moments<<<nblk, 256, 0, c->stream>>>(ra.gram, mu, P, M, 1);
    else if (mode == kModeHund1) finalize_moments_ph<<<nblk, 256, 0, c->stream>>>(ra.gram, mu, ra.sites, P, Ps, M, 1, c->p.L);
    else finalize_moments_dex<<<nblk, 256, 0, c->stream>>>(ra.gram, mu, c->ptr<double>(c->lay.vnorm2), P, Ps, M, 1);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return GFMC_OK;
}

// a2 + a3 + moment read-out with TWO Chebyshev steps per pass (cheb_step2.cuh; one-vector mode, L = 32, M/2 even): M/4 launches.
int run_moments_two_step(gfmc_ctx* c, int P)
{
    const int L = c->p.L, M = c->p.M;
    const int Ps = slots_of(kModeHund1, P);
    const int ntiles = 2;
    if ((size_t)Ps * ntiles * 8 > c->lay.gram_doubles_per_step) return fail(c, GFMC_ENOMEM, "gram scratch too small");
    const int32_t* sites = c->ptr<int32_t>(c->lay.sites);
    double2* R[4] = {c->ptr<double2>(c->lay.R0), c->ptr<double2>(c->lay.R1), c->ptr<double2>(c->lay.R2), c->ptr<double2>(c->lay.R3)};
    CU_TRY(c, cudaMemsetAsync(R[0], 0, (size_t)32 * c->N * P, c->stream));
    init_start_vectors_ph2<<<(P + 255) / 256, 256, 0, c->stream>>>(R[0], sites, P, L);
    c->counts[1] += 1;
    auto* ev = next_timing_events(c);
    if (ev) CU_TRY(c, cudaEventRecord(ev->first, c->stream));
    Step2Args sa{};
    sa.Sx = c->ptr<double>(c->lay.Sx); sa.Sy = c->ptr<double>(c->lay.Sy); sa.Sz = c->ptr<double>(c->lay.Sz);
    sa.P = P; sa.nitems = 2 * P;
    double* gram = c->ptr<double>(c->lay.gram);
    const size_t gstride = (size_t)Ps * ntiles * 8;
    const double ta = c->p.t / c->a, ja = c->p.JH / c->a;
    const unsigned grid = (unsigned)std::min(sa.nitems, c->nSM);
    const int npass = M / 4;
    for (int k = 1; k <= npass; ++k) {
        // pass 1: r_0 = R0 -> (r_1, r_2) = (R1, R2); even passes: (R1, R2) -> (R3, R0); odd passes >= 3: (R3, R0) -> (R1, R2)
        if (k == 1) { sa.prv = nullptr; sa.cur = R[0]; sa.out1 = R[1]; sa.out2 = R[2]; }
        else if ((k & 1) == 0) { sa.prv = R[1]; sa.cur = R[2]; sa.out1 = R[3]; sa.out2 = R[0]; }
        else { sa.prv = R[3]; sa.cur = R[0]; sa.out1 = R[1]; sa.out2 = R[2]; }
        const double s1 = (k == 1) ? 1.0 : 2.0;
        sa.ct1 = -s1 * ta; sa.cj1 = s1 * ja; sa.ct2 = -2.0 * ta; sa.cj2 = 2.0 * ja;
        sa.gram1 = gram + (size_t)(2 * k - 2) * gstride; sa.gram2 = gram + (size_t)(2 * k - 1) * gstride;
        if (k == 1) cheb_step2_kernel<true><<<grid, k2Threads, k2SmemBytes, c->stream>>>(sa);
        else cheb_step2_kernel<false><<<grid, k2Threads, k2SmemBytes, c->stream>>>(sa);
    }
    c->counts[0] += npass;
    if (ev) { c->loop_steps += M / 2; CU_TRY(c, cudaEventRecord(ev->second, c->stream)); }     // fused STEPS, two per launch
    c->loop_vectors = (int64_t)P;
    const long long nthreads = (long long)P * (M / 2 + 1);
    finalize_moments_ph<<<(unsigned)((nthreads + 255) / 256), 256, 0, c->stream>>>(gram, c->ptr<double2>(c->lay.mu), sites, P, Ps, M, ntiles, L);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return GFMC_OK;
}

// a2 + a3 + moment read-out for the P sites already stored in ctx->sites (device).  Leaves mu [P][M][4] on the device.
// prop_dev / by_site: trial spins (kModeDex only: |v> of Eq. (21) depends on S'_o).
int run_moments_batch(gfmc_ctx* c, int P, const double* prop_dev, int by_site)
{
    const int L = c->p.L, M = c->p.M, mode = c->mode;
    const int NG = gram_width(mode);
    const int Ps = slots_of(mode, P);
    StepPlan pl = make_plan(L, Ps, c->nSM, c->smem_limit, NG, c->tun);
    if (!pl.ok) return fail(c, GFMC_EINVAL, "no launch plan for L=%d slots=%d", L, Ps);
    if ((size_t)Ps * pl.ntiles * NG > c->lay.gram_doubles_per_step) return fail(c, GFMC_ENOMEM, "gram scratch too small");
    if (mode == kModeDex && !prop_dev) return fail(c, GFMC_EINVAL, "the J_H->inf model needs the trial spins to build |v> (Eq. 21)");
    const int32_t* sites = c->ptr<int32_t>(c->lay.sites);
    if (c->tun.two_step) return run_moments_two_step(c, P);
    const ResidentPlan rp = make_resident_plan(L, c->smem_limit, c->tun);
    if (rp.ok) return run_moments_resident(c, P, Ps, rp, prop_dev, by_site);
    // explicit work list (balanced ranges of planes per CTA) where the arithmetic enumeration would waste part of the last round
    const bool streamk = streamk_applicable(pl, L, c->nSM, c->tun.streamk_eff);
    int sk_which = 0;
    if (streamk) {
        int rc = upload_item_table(c, pl, Ps, &sk_which); if (rc) return rc;
        pl.ntiles = c->sk[sk_which].ntiles; pl.grid = c->nSM;
        if ((size_t)Ps * pl.ntiles * NG > c->lay.gram_doubles_per_step) return fail(c, GFMC_ENOMEM, "gram scratch too small");
        // a column that is not cut has only its first tile written: the second must read as zero
        CU_TRY(c, cudaMemsetAsync(c->ptr<double>(c->lay.gram), 0, (size_t)(M / 2) * Ps * pl.ntiles * NG * sizeof(double), c->stream));
    }
    double2* R[2] = {c->ptr<double2>(c->lay.R0), c->ptr<double2>(c->lay.R1)};
    const size_t rbytes = (size_t)64 * c->N * Ps;
    CU_TRY(c, cudaMemsetAsync(R[0], 0, rbytes, c->stream));
    if (mode == kModeHund2) init_start_vectors<<<(P + 255) / 256, 256, 0, c->stream>>>(R[0], sites, P, L);
    else if (mode == kModeHund1) init_start_vectors_ph<<<(P + 255) / 256, 256, 0, c->stream>>>(R[0], sites, P, Ps, L);
    else init_start_vectors_dex<<<(P + 127) / 128, 128, 0, c->stream>>>(R[0], sites, prop_dev, by_site, c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy),
                                                                       c->ptr<double>(c->lay.Sz), c->p.t, c->ptr<double>(c->lay.vnorm2), P, Ps, L);
    c->counts[1] += 1;

    auto* ev = next_timing_events(c);
    if (ev) CU_TRY(c, cudaEventRecord(ev->first, c->stream));

    StepArgs sa{};
    sa.Sx = c->ptr<double>(c->lay.Sx); sa.Sy = c->ptr<double>(c->lay.Sy); sa.Sz = c->ptr<double>(c->lay.Sz);
    sa.Tx = c->ptr<double2>(c->lay.Tx); sa.Ty = c->ptr<double2>(c->lay.Ty); sa.Tz = c->ptr<double2>(c->lay.Tz);
    sa.Tq = c->ptr<double2>(c->lay.Tq); sa.nst_t = pl.nst_t; sa.tstage_units = pl.tstage_units;
    sa.L = L; sa.P = Ps; sa.full = pl.full; sa.G = pl.G; sa.Ty_rows = pl.Ty; sa.nty = pl.nty; sa.nzc = pl.nzc; sa.nzper = pl.nzper;
    sa.nitems = pl.nitems; sa.nst_c = pl.nst_c; sa.nst_p = pl.nst_p; sa.cstage_units = pl.cstage_units; sa.pstage_units = pl.pstage_units;
    sa.slow_reduce = pl.slow_reduce;
    sa.items = nullptr; sa.cta_start = nullptr; sa.ntiles = pl.ntiles;
    if (streamk) {
        sa.items = c->ptr<WorkItem>(c->lay.items) + (size_t)sk_which * c->lay.max_items;
        sa.cta_start = c->ptr<int>(c->lay.cta_start) + (size_t)sk_which * (c->nSM + 2);
        sa.ntiles = pl.ntiles;
    }
    double* gram = c->ptr<double>(c->lay.gram);
    const size_t gstride = (size_t)Ps * pl.ntiles * NG;
    const double JH = (mode == kModeDex) ? 0.0 : c->p.JH;
    for (int m = 1; m <= M / 2; ++m) {
        sa.cur = R[(m - 1) & 1];
        sa.nxt = R[m & 1];
        sa.gram = gram + (size_t)(m - 1) * gstride;
        const double scale = (m == 1) ? 1.0 : 2.0;
        sa.ct = -scale * c->p.t / c->a;
        sa.cj = scale * JH / c->a;
        launch_step(mode, L, m == 1, pl, sa, c->stream);
    }
    c->counts[0] += M / 2;
    if (ev) c->loop_steps += M / 2;
    c->loop_vectors = (mode == kModeHund1) ? (int64_t)P : 2 * (int64_t)P;
    if (ev) CU_TRY(c, cudaEventRecord(ev->second, c->stream));
    const long long nthreads = (long long)P * (M / 2 + 1);
    const unsigned nblk = (unsigned)((nthreads + 255) / 256);
    double2* mu = c->ptr<double2>(c->lay.mu);
    if (mode == kModeHund2) finalize_moments<<<nblk, 256, 0, c->stream>>>(gram, mu, P, M, pl.ntiles);
    else if (mode == kModeHund1) finalize_moments_ph<<<nblk, 256, 0, c->stream>>>(gram, mu, sites, P, Ps, M, pl.ntiles, L);
    else finalize_moments_dex<<<nblk, 256, 0, c->stream>>>(gram, mu, c->ptr<double>(c->lay.vnorm2), P, Ps, M, pl.ntiles);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return GFMC_OK;
}

size_t green_smem_bytes(const gfmc_ctx* c, int Mc) { return (size_t)Mc * 4 * 16 + (size_t)c->K * 16 + (size_t)c->K * 8; }

// a4-a6 for the P sites in ctx->sites whose moments are in ctx->mu.
int run_green(gfmc_ctx* c, int first, int P, double2* G_out, const double* proposals_dev, int by_site, double* dS_dev)
{
    GreenArgs ga{};
    ga.mu = c->ptr<double2>(c->lay.mu) + (size_t)first * c->p.M * 4;
    ga.w = c->ptr<double>(c->lay.w);
    ga.tw = c->ptr<double2>(c->lay.tw);
    ga.G = G_out;
    ga.sites = c->ptr<int32_t>(c->lay.sites) + first;
    ga.Sx = c->ptr<double>(c->lay.Sx); ga.Sy = c->ptr<double>(c->lay.Sy); ga.Sz = c->ptr<double>(c->lay.Sz);
    ga.proposals = proposals_dev; ga.dS = dS_dev; ga.by_site = by_site; ga.dex = (c->mode == kModeDex);
    ga.n = P; ga.M = c->p.M; ga.K = c->K; ga.Mc = std::min(c->p.M, 1024);
    ga.a = c->a; ga.b = c->b; ga.JH = c->p.JH; ga.beta = 1.0 / c->p.T; ga.mu_chem = c->p.mu;
    // a5 by FFT (f4) when the node count is a power of two and work[2K] + out[4][K] fit in shared memory; else the direct sum
    const size_t fft_bytes = (size_t)6 * c->K * 16;
    const bool use_fft = !c->tun.green_direct && c->K >= 64 && (c->K & (c->K - 1)) == 0 && fft_bytes + 4096 <= c->smem_limit;
    if (use_fft) green_fft_dS_kernel<<<P, kGreenThreads, fft_bytes, c->stream>>>(ga);
    else green_dS_kernel<<<P, kGreenThreads, green_smem_bytes(c, ga.Mc), c->stream>>>(ga);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return GFMC_OK;
}

// f5: one batch decided sequentially and exactly (exact_batch.cuh) for the P sites in ctx->sites: plain recursion (M-1 fused steps,
// cross moments read out after every step), Green blocks between all pairs of sites, then per site: decision kernel + Woodbury
// update of the later blocks.  Always the streaming kernel (the read-out needs the vectors in global memory after every step).
int run_exact_batch(gfmc_ctx* c, int P, const double* prop_dev, const double* uni_dev, int by_site,
                    uint8_t* accepted_dev, double* dS_log_dev, uint8_t* acc_log_dev, unsigned long long* counter_dev)
{
    const int L = c->p.L, M = c->p.M, K = c->K;
    if (c->mode != kModeHund2 || c->p.exact_batch_sites <= 0)
        return fail(c, GFMC_ESTATE, "exact batches need a context created with exact_batch_sites > 0 (Eq. (1) model, ph_symmetry = 0)");
    if (P > c->p.exact_batch_sites) return fail(c, GFMC_EINVAL, "exact batch of %d sites > exact_batch_sites %d", P, c->p.exact_batch_sites);
    StepPlan pl = make_plan(L, P, c->nSM, c->smem_limit, 8, c->tun);
    if (!pl.ok) return fail(c, GFMC_EINVAL, "no launch plan for L=%d slots=%d", L, P);
    if ((size_t)P * pl.ntiles * 8 > c->lay.gram_doubles_per_step) return fail(c, GFMC_ENOMEM, "gram scratch too small");
    const int32_t* sites = c->ptr<int32_t>(c->lay.sites);
    double2* R[2] = {c->ptr<double2>(c->lay.R0), c->ptr<double2>(c->lay.R1)};
    double2* xmu = c->ptr<double2>(c->lay.xmu);
    double2* xG = c->ptr<double2>(c->lay.xG);
    CU_TRY(c, cudaMemsetAsync(R[0], 0, (size_t)64 * c->N * P, c->stream));
    init_start_vectors<<<(P + 255) / 256, 256, 0, c->stream>>>(R[0], sites, P, L);
    const unsigned rb = (unsigned)((P * P * 4 + 255) / 256);
    cross_readout_kernel<<<rb, 256, 0, c->stream>>>(R[0], sites, P, L, M, 0, xmu);
    c->counts[1] += 2;
    auto* ev = next_timing_events(c);
    if (ev) CU_TRY(c, cudaEventRecord(ev->first, c->stream));
    StepArgs sa{};
    sa.Sx = c->ptr<double>(c->lay.Sx); sa.Sy = c->ptr<double>(c->lay.Sy); sa.Sz = c->ptr<double>(c->lay.Sz);
    sa.L = L; sa.P = P; sa.full = pl.full; sa.G = pl.G; sa.Ty_rows = pl.Ty; sa.nty = pl.nty; sa.nzc = pl.nzc; sa.nzper = pl.nzper;
    sa.nitems = pl.nitems; sa.nst_c = pl.nst_c; sa.nst_p = pl.nst_p; sa.cstage_units = pl.cstage_units; sa.pstage_units = pl.pstage_units;
    sa.slow_reduce = pl.slow_reduce; sa.items = nullptr; sa.cta_start = nullptr; sa.ntiles = pl.ntiles;
    sa.gram = c->ptr<double>(c->lay.gram);             // the Gram sums of the fused step are not used in this mode: one scratch slice
    for (int m = 1; m < M; ++m) {
        sa.cur = R[(m - 1) & 1];
        sa.nxt = R[m & 1];
        const double scale = (m == 1) ? 1.0 : 2.0;
        sa.ct = -scale * c->p.t / c->a;
        sa.cj = scale * c->p.JH / c->a;
        launch_step(kModeHund2, L, m == 1, pl, sa, c->stream);
        cross_readout_kernel<<<rb, 256, 0, c->stream>>>(R[m & 1], sites, P, L, M, m, xmu);
    }
    c->counts[0] += M - 1; c->counts[1] += M - 1;
    if (ev) { c->loop_steps += M - 1; CU_TRY(c, cudaEventRecord(ev->second, c->stream)); }
    c->loop_vectors = 2 * (int64_t)P;
    // Green blocks of all P*P pairs (physical units) by the same reconstruction kernels as the diagonal blocks
    {
        GreenArgs ga{};
        ga.mu = xmu; ga.w = c->ptr<double>(c->lay.w); ga.tw = c->ptr<double2>(c->lay.tw); ga.G = xG; ga.sites = sites;
        ga.Sx = sa.Sx; ga.Sy = sa.Sy; ga.Sz = sa.Sz; ga.proposals = nullptr; ga.dS = nullptr; ga.by_site = 0; ga.dex = 0;
        ga.n = P * P; ga.M = M; ga.K = K; ga.Mc = std::min(M, 1024);
        ga.a = c->a; ga.b = c->b; ga.JH = c->p.JH; ga.beta = 1.0 / c->p.T; ga.mu_chem = c->p.mu;
        const size_t fft_bytes = (size_t)6 * K * 16;
        const bool use_fft = !c->tun.green_direct && K >= 64 && (K & (K - 1)) == 0 && fft_bytes + 4096 <= c->smem_limit;
        if (use_fft) green_fft_dS_kernel<<<P * P, kGreenThreads, fft_bytes, c->stream>>>(ga);
        else green_dS_kernel<<<P * P, kGreenThreads, green_smem_bytes(c, ga.Mc), c->stream>>>(ga);
        c->counts[1] += 1;
    }
    ExactArgs ea{};
    ea.G = xG; ea.sites = sites; ea.proposals = prop_dev; ea.uniforms = uni_dev; ea.by_site = by_site;
    ea.Sx = c->ptr<double>(c->lay.Sx); ea.Sy = c->ptr<double>(c->lay.Sy); ea.Sz = c->ptr<double>(c->lay.Sz);
    ea.dS = c->ptr<double>(c->lay.dS); ea.accepted = accepted_dev ? accepted_dev : c->ptr<uint8_t>(c->lay.acc);
    ea.dS_log = dS_log_dev; ea.accept_log = acc_log_dev; ea.n_accepted = counter_dev;
    ea.P = P; ea.K = K; ea.a = c->a; ea.b = c->b; ea.JH = c->p.JH; ea.beta = 1.0 / c->p.T; ea.mu_chem = c->p.mu;
    ea.bad = reinterpret_cast<unsigned int*>(c->ptr<unsigned long long>(c->lay.scal) + 20);
    CU_TRY(c, cudaMemsetAsync(ea.bad, 0, sizeof(unsigned int), c->stream));
    for (int j = 0; j < P; ++j) {
        ea.j = j;
        exact_decide_kernel<<<1, kGreenThreads, (size_t)K * 24, c->stream>>>(ea);
        c->counts[1] += 1;
        const long long work = (long long)(P - j - 1) * (P - j - 1) * K;
        if (work > 0) {
            exact_update_kernel<<<(unsigned)((work + 255) / 256), 256, 0, c->stream>>>(ea);
            c->counts[1] += 1;
        }
    }
    // A node where d_k = det(1 + G_jj Delta_j) vanishes (or a NaN that came in through unvalidated device inputs) has no Woodbury
    // update, and every later decision of the batch would compare NaN with ln u and read as "rejected".  Say so instead: the batch
    // is abandoned BEFORE any flip is written, the configuration stays as it was at batch start.
    unsigned int bad = 0;
    CU_TRY(c, cudaMemcpyAsync(&bad, ea.bad, sizeof bad, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    if (bad)
        return fail(c, GFMC_ESTATE, "exact batch abandoned, configuration unchanged: %s%s%s", (bad & 1u) ? "non-finite Delta S" : "",
                    bad == 3u ? " and " : "", (bad & 2u) ? "singular 1 + G Delta at an energy node (d_k = 0)" : "");
    exact_apply_kernel<<<(P + 127) / 128, 128, 0, c->stream>>>(ea);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return GFMC_OK;
}

int check_sites_host(gfmc_ctx* c, const int32_t* sites, int n)
{
    for (int i = 0; i < n; ++i)
        if (sites[i] < 0 || sites[i] >= c->N) return fail(c, GFMC_EINVAL, "site %d out of range at position %d", sites[i], i);
    return GFMC_OK;
}

}  // namespace

extern "C" {

const char* gfmc_version(void) { return "gfmc-b200 0.1 (sm_100a)"; }
const char* gfmc_create_error(void) { return g_create_error.c_str(); }

size_t gfmc_workspace_bytes(const gfmc_params* params)
{
    if (!valid_params(params)) return 0;
    // sized with the properties of the device the context will live on (exactly what gfmc_create does); only without any CUDA
    // device (sizing on a build host) the B200 values are assumed: 148 SMs, 227 KiB of opt-in shared memory per CTA
    int nSM = 148; size_t smem = 232448;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) == cudaSuccess && params->device >= 0 && params->device < ndev) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, params->device) == cudaSuccess && v > 0) nSM = v;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, params->device) == cudaSuccess && v > 0) smem = (size_t)v;
    } else (void)cudaGetLastError();
    return make_layout(params, nSM, smem).total;
}

int gfmc_create(const gfmc_params* params, gfmc_ctx** out)
{
    if (!out) return fail(nullptr, GFMC_EINVAL, "out is NULL");
    *out = nullptr;
    if (!valid_params(params)) return fail(nullptr, GFMC_EINVAL, "invalid parameters (L in [2,256], M even >= 2, T > 0, kernel in 0..2, max_batch_sites >= 1)");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, GFMC_ECUDA, "no CUDA device: %s (libgfmc has no CPU fallback)", e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    if (params->device < 0 || params->device >= ndev) return fail(nullptr, GFMC_EINVAL, "device %d out of range", params->device);
    if ((e = cudaSetDevice(params->device)) != cudaSuccess) return fail(nullptr, GFMC_ECUDA, "cudaSetDevice: %s", cudaGetErrorString(e));
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, params->device)) != cudaSuccess) return fail(nullptr, GFMC_ECUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e));
    if (prop.major != 10) return fail(nullptr, GFMC_ECUDA, "device is sm_%d%d; libgfmc is built for sm_100a only", prop.major, prop.minor);

    gfmc_ctx* c = new (std::nothrow) gfmc_ctx();
    if (!c) return fail(nullptr, GFMC_ENOMEM, "host allocation failed");
    c->p = *params;
    c->tun = tuning_of(params);
    c->N = params->L * params->L * params->L;
    c->D = 2 * c->N;
    c->K = params->n_energy > 0 ? params->n_energy : 2 * params->M;
    c->p.n_energy = c->K;
    c->mode = mode_of(params);
    // a1: spin-independent Gershgorin bounds.  Eq. (1): 6|t| + sqrt(2)|J_H|;  Eq. (2)-(3): |t_ij| <= 1, so 6|t|.
    c->a = (c->mode == kModeDex) ? 6.0 * std::fabs(params->t) : 6.0 * std::fabs(params->t) + std::sqrt(2.0) * std::fabs(params->JH);
    c->b = 0.0;
    c->lambda = params->lambda > 0.0 ? params->lambda : 4.0;
    c->stream = reinterpret_cast<cudaStream_t>(params->stream);
    c->nSM = prop.multiProcessorCount;
    c->smem_limit = prop.sharedMemPerBlockOptin;
    c->spins_set = false;
    c->counts[0] = c->counts[1] = 0;
    c->ev_used = 0; c->loop_steps = 0; c->loop_vectors = 0; c->loop_ms = 0.0;
    c->pinned = nullptr; c->pinned_bytes = 0;
    c->capturing = false;
    c->own_stream = false;
    c->sk[0] = c->sk[1] = gfmc_ctx::WorkList{0, 0, 0}; c->sk_clock = 0; c->graph_clock = 0;
    c->run_sweeps = 0; c->batch_mode = GFMC_BATCH_FROZEN;
    c->throttle_ev[0] = c->throttle_ev[1] = nullptr; c->throttle_n = 0;
    c->lay = make_layout(&c->p, c->nSM, c->smem_limit);

    auto bail = [&](int code, const std::string& msg) { g_create_error = msg; gfmc_destroy(c); return code; };

    if (!make_plan(params->L, slots_of(c->mode, params->max_batch_sites), c->nSM, c->smem_limit, gram_width(c->mode), c->tun).ok)
        return bail(GFMC_EINVAL, "lattice edge too large for the shared-memory ring");
    if (green_smem_bytes(c, std::min(params->M, 1024)) + 4096 > c->smem_limit)
        return bail(GFMC_EINVAL, "n_energy too large for the Green-function kernel's shared memory");
    if (params->workspace) {
        if (params->workspace_bytes < c->lay.total) return bail(GFMC_ENOMEM, "workspace too small");
        if (reinterpret_cast<uintptr_t>(params->workspace) % 256) return bail(GFMC_EINVAL, "workspace not 256-byte aligned");
        c->arena = static_cast<char*>(params->workspace); c->own_arena = false;
    } else {
        void* ptr = nullptr;
        if ((e = cudaMalloc(&ptr, c->lay.total)) != cudaSuccess) {
            (void)cudaGetLastError();
            char buf[160]; snprintf(buf, sizeof buf, "cudaMalloc of %zu bytes failed: %s", c->lay.total, cudaGetErrorString(e));
            return bail(GFMC_ENOMEM, buf);
        }
        c->arena = static_cast<char*>(ptr); c->own_arena = true;
    }
    // opt in to large dynamic shared memory
    if (!c->stream) {
        // NULL means "the legacy default stream" to the caller.  The context runs on its own non-blocking stream instead: every call
        // first waits for what is queued on the legacy stream (begin_call) and synchronises its stream before returning, so the
        // ordering the caller sees is that of the legacy stream -- but contexts do not serialise each other, and the stream can be
        // captured into CUDA graphs.
        if ((e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaEventCreateWithFlags(&c->legacy_ev, cudaEventDisableTiming)) != cudaSuccess)
            return bail(GFMC_ECUDA, std::string("cudaStreamCreate: ") + cudaGetErrorString(e));
        c->own_stream = true;
    }
    e = set_step_smem_limit((int)c->smem_limit);
    if (e == cudaSuccess) e = set_resident_smem_limit_mode<kModeHund2>((int)c->smem_limit);
    if (e == cudaSuccess) e = set_resident_smem_limit_mode<kModeHund1>((int)c->smem_limit);
    if (e == cudaSuccess) e = set_resident_smem_limit_mode<kModeDex>((int)c->smem_limit);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(green_dS_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_limit - 4096);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(green_fft_dS_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_limit - 4096);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_step2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k2SmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(cheb_step2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k2SmemBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(exact_decide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_limit - 4096);
    {
        // every kernel of the per-batch sequence asks for the same (maximum shared memory) L1/shared split, so that alternating
        // between them -- in one chain or across concurrently running contexts -- never forces an SM to drain and reconfigure
        const int co = cudaSharedmemCarveoutMaxShared;
        const void* fns[] = {(const void*)next_batch_kernel, (const void*)finalize_moments, (const void*)finalize_moments_ph, (const void*)finalize_moments_dex,
                             (const void*)init_start_vectors_dex, (const void*)dex_bonds_kernel, (const void*)green_dS_kernel, (const void*)green_fft_dS_kernel,
                             (const void*)metropolis_kernel, (const void*)propose_kernel, (const void*)magnetization_kernel,
                             (const void*)cheb_resident_kernel<kModeHund2, 1>, (const void*)cheb_resident_kernel<kModeHund1, 1>, (const void*)cheb_resident_kernel<kModeDex, 1>,
                             (const void*)cheb_resident_kernel<kModeHund2, 2>, (const void*)cheb_resident_kernel<kModeHund1, 2>, (const void*)cheb_resident_kernel<kModeDex, 2>,
                             (const void*)cheb_resident_kernel<kModeHund2, 3>, (const void*)cheb_resident_kernel<kModeHund1, 3>, (const void*)cheb_resident_kernel<kModeDex, 3>,
                             (const void*)cheb_resident_kernel<kModeHund2, 4>, (const void*)cheb_resident_kernel<kModeHund1, 4>, (const void*)cheb_resident_kernel<kModeDex, 4>};
        for (const void* f : fns)
            if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, co);
    }
    if (e != cudaSuccess) return bail(GFMC_ECUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e));

    // tables (host libm, uploaded once): damping weights w_m (a4) and twiddles exp(-i pi p / (2K)) (a5)
    const int M = params->M, K = c->K;
    std::vector<double> w(M);
    const double pi = 3.141592653589793238462643383279502884;
    for (int m = 0; m < M; ++m) {
        double g;
        if (params->kernel == GFMC_KERNEL_JACKSON) {
            const double q = pi / (M + 1.0);
            g = ((M - m + 1.0) * std::cos(q * m) + std::sin(q * m) / std::tan(q)) / (M + 1.0);
        } else if (params->kernel == GFMC_KERNEL_LORENTZ) {
            g = std::sinh(c->lambda * (1.0 - (double)m / M)) / std::sinh(c->lambda);
        } else g = 1.0;
        w[m] = (m == 0) ? 0.5 * g : g;
    }
    std::vector<double> tw((size_t)8 * K);
    for (int p = 0; p < 4 * K; ++p) {
        const double ang = pi * (double)p / (2.0 * K);
        tw[2 * (size_t)p] = std::cos(ang); tw[2 * (size_t)p + 1] = -std::sin(ang);
    }
    // colour-major site order (O5 schedule)
    c->order_h.resize(c->N);
    int n = 0;
    const int L = params->L;
    for (int col = 0; col < 2; ++col) {
        int cnt = 0;
        for (int i = 0; i < c->N; ++i) {
            const int x = i % L, y = (i / L) % L, z = i / (L * L);
            if (((x + y + z) & 1) == col) { c->order_h[n++] = i; ++cnt; }
        }
        c->ncolour[col] = cnt;
    }
    if ((e = cudaMemcpyAsync(c->ptr<double>(c->lay.w), w.data(), (size_t)M * 8, cudaMemcpyHostToDevice, c->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(c->ptr<double>(c->lay.tw), tw.data(), tw.size() * 8, cudaMemcpyHostToDevice, c->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(c->ptr<int32_t>(c->lay.order), c->order_h.data(), (size_t)c->N * 4, cudaMemcpyHostToDevice, c->stream)) != cudaSuccess ||
        (e = cudaStreamSynchronize(c->stream)) != cudaSuccess)
        return bail(GFMC_ECUDA, std::string("table upload: ") + cudaGetErrorString(e));
    *out = c;
    return GFMC_OK;
}

int gfmc_destroy(gfmc_ctx* c)
{
    if (!c) return GFMC_OK;
    cudaSetDevice(c->p.device);
    cudaStreamSynchronize(c->stream);
    for (auto& ev : c->ev_pool) { cudaEventDestroy(ev.first); cudaEventDestroy(ev.second); }
    for (auto& gr : c->graphs) cudaGraphExecDestroy(gr.exec);
    for (auto& te : c->throttle_ev) if (te) cudaEventDestroy(te);
    if (c->own_stream) { cudaStreamDestroy(c->stream); cudaEventDestroy(c->legacy_ev); }
    if (c->own_arena && c->arena) cudaFree(c->arena);
    if (c->pinned) cudaFreeHost(c->pinned);
    delete c;
    return GFMC_OK;
}

const char* gfmc_last_error(const gfmc_ctx* c) { return c ? c->err.c_str() : "NULL context"; }

int gfmc_bounds(const gfmc_ctx* c, double* a, double* b)
{
    if (!c || !a || !b) return GFMC_EINVAL;
    *a = c->a; *b = c->b;
    return GFMC_OK;
}

int gfmc_launch_counts(const gfmc_ctx* c, int64_t counts[2])
{
    if (!c || !counts) return GFMC_EINVAL;
    counts[0] = c->counts[0]; counts[1] = c->counts[1];
    return GFMC_OK;
}

int gfmc_last_step_loop_ms(const gfmc_ctx* c, double* ms, int64_t* n_steps)
{
    if (!c) return GFMC_EINVAL;
    if (ms) *ms = c->loop_ms;
    if (n_steps) *n_steps = c->loop_steps;
    return GFMC_OK;
}

int gfmc_last_step_loop_vectors(const gfmc_ctx* c, int64_t* n_vectors, int64_t* bytes_per_step)
{
    if (!c) return GFMC_EINVAL;
    if (n_vectors) *n_vectors = c->loop_vectors;
    // algorithmic bytes of one fused step: 48 B per complex element of every start vector that is propagated
    if (bytes_per_step) *bytes_per_step = 48 * c->loop_vectors * (c->mode == kModeDex ? (int64_t)c->N : (int64_t)c->D);
    return GFMC_OK;
}

int gfmc_set_spins(gfmc_ctx* c, const double* S, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_set_spins");
    if (!S || (mem != GFMC_HOST && mem != GFMC_DEVICE)) return fail(c, GFMC_EINVAL, "gfmc_set_spins: bad argument");
    CU_TRY(c, cudaSetDevice(c->p.device));
    if (mem == GFMC_HOST) {
        for (int i = 0; i < c->N; ++i) {
            const double n2 = S[3 * i] * S[3 * i] + S[3 * i + 1] * S[3 * i + 1] + S[3 * i + 2] * S[3 * i + 2];
            if (!(std::fabs(std::sqrt(n2) - 1.0) <= 1e-12)) return fail(c, GFMC_EINVAL, "spin %d is not a unit vector (|S| = %.17g)", i, std::sqrt(n2));
        }
    }
    double* aos = c->ptr<double>(c->lay.Saos);
    int rc = copy_in(c, aos, S, (size_t)24 * c->N, mem);
    if (rc) return rc;
    spins_aos_to_soa<<<(c->N + 255) / 256, 256, 0, c->stream>>>(aos, c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy), c->ptr<double>(c->lay.Sz), c->N);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    rc = refresh_bonds(c);
    if (rc) return rc;
    rc = guard.finish();
    if (rc == GFMC_OK) c->spins_set = true;
    return rc;
}

int gfmc_get_spins(gfmc_ctx* c, double* S, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_get_spins");
    if (!S || (mem != GFMC_HOST && mem != GFMC_DEVICE)) return fail(c, GFMC_EINVAL, "gfmc_get_spins: bad argument");
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "spins not set");
    CU_TRY(c, cudaSetDevice(c->p.device));
    double* aos = c->ptr<double>(c->lay.Saos);
    spins_soa_to_aos<<<(c->N + 255) / 256, 256, 0, c->stream>>>(c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy), c->ptr<double>(c->lay.Sz), aos, c->N);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    int rc = copy_out(c, S, aos, (size_t)24 * c->N, mem);
    if (rc) return rc;
    return guard.finish();
}

int gfmc_magnetization(gfmc_ctx* c, double* m)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_magnetization");
    if (!m) return fail(c, GFMC_EINVAL, "gfmc_magnetization: NULL output");
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "spins not set");
    CU_TRY(c, cudaSetDevice(c->p.device));
    double* scal = c->ptr<double>(c->lay.scal);
    magnetization_kernel<<<1, 1024, 0, c->stream>>>(c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy), c->ptr<double>(c->lay.Sz), c->N, scal,
                                                    nullptr, nullptr);
    c->counts[1] += 1;
    CU_TRY(c, cudaMemcpyAsync(m, scal, 8, cudaMemcpyDeviceToHost, c->stream));
    return guard.finish();
}

// shared front end of gfmc_moments / gfmc_local_green / gfmc_delta_S: loops over chunks of max_batch_sites.
// proposals [n_sites][3] (may be NULL for the Eq. (1) model) are staged chunk by chunk into ctx->prop.
static int for_chunks(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, int mem, const char* who,
                      int (*body)(gfmc_ctx*, int first, int P, void* user), void* user)
{
    if (!sites || n_sites < 0 || (mem != GFMC_HOST && mem != GFMC_DEVICE)) return fail(c, GFMC_EINVAL, "%s: bad argument", who);
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "%s: spins not set", who);
    if (c->mode == kModeDex && !proposals) return fail(c, GFMC_EINVAL, "%s: the J_H->inf model needs trial spins (use the _ov entry points)", who);
    CU_TRY(c, cudaSetDevice(c->p.device));
    if (mem == GFMC_HOST) { int rc = check_sites_host(c, sites, n_sites); if (rc) return rc; }
    const int B = c->p.max_batch_sites;
    for (int first = 0; first < n_sites; first += B) {
        const int P = std::min(B, n_sites - first);
        int rc = copy_in(c, c->ptr<int32_t>(c->lay.sites), sites + first, (size_t)P * 4, mem);
        if (rc) return rc;
        if (proposals) { rc = copy_in(c, c->ptr<double>(c->lay.prop), proposals + (size_t)first * 3, (size_t)P * 24, mem); if (rc) return rc; }
        rc = run_moments_batch(c, P, proposals ? c->ptr<double>(c->lay.prop) : nullptr, 0);
        if (rc) return rc;
        rc = body(c, first, P, user);
        if (rc) return rc;
    }
    return GFMC_OK;
}

struct MomentsUser { double* mu; int mem; };
static int moments_impl(gfmc_ctx* c, CallGuard& guard, const int32_t* sites, int32_t n_sites, const double* proposals, double* mu, int mem, const char* who)
{
    if (!mu) return fail(c, GFMC_EINVAL, "%s: NULL output", who);
    MomentsUser u{mu, mem};
    int rc = for_chunks(c, sites, n_sites, proposals, mem, who, [](gfmc_ctx* c, int first, int P, void* user) {
        auto* u = static_cast<MomentsUser*>(user);
        const size_t per = (size_t)c->p.M * 4 * 16;
        return copy_out(c, reinterpret_cast<char*>(u->mu) + (size_t)first * per, c->ptr<char>(c->lay.mu), (size_t)P * per, u->mem);
    }, &u);
    if (rc) return rc;
    return guard.finish();
}

int gfmc_moments(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, double* mu, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_moments");
    if (c->mode == kModeDex) return fail(c, GFMC_EINVAL, "gfmc_moments: model is GFMC_MODEL_DEX_INF, use gfmc_moments_ov");
    return moments_impl(c, guard, sites, n_sites, nullptr, mu, mem, "gfmc_moments");
}

int gfmc_moments_ov(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, double* mu, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_moments_ov");
    if (c->mode != kModeDex) return fail(c, GFMC_EINVAL, "gfmc_moments_ov: model is GFMC_MODEL_HUND, use gfmc_moments");
    if (!proposals) return fail(c, GFMC_EINVAL, "gfmc_moments_ov: NULL proposals");
    return moments_impl(c, guard, sites, n_sites, proposals, mu, mem, "gfmc_moments_ov");
}

struct GreenUser { double* G; int mem; };
static int green_impl(gfmc_ctx* c, CallGuard& guard, const int32_t* sites, int32_t n_sites, const double* proposals, double* E, double* G, int mem, const char* who)
{
    if (E) {
        // E_k = a cos(pi (k + 1/2)/K) + b
        std::vector<double> Eh(c->K);
        const double pi = 3.141592653589793238462643383279502884;
        for (int k = 0; k < c->K; ++k) Eh[k] = c->a * std::cos(pi * (k + 0.5) / c->K) + c->b;
        if (mem == GFMC_HOST) std::memcpy(E, Eh.data(), (size_t)c->K * 8);
        else { CU_TRY(c, cudaMemcpyAsync(E, Eh.data(), (size_t)c->K * 8, cudaMemcpyHostToDevice, c->stream)); CU_TRY(c, cudaStreamSynchronize(c->stream)); }
    }
    if (!G) return (n_sites == 0 || sites) ? GFMC_OK : fail(c, GFMC_EINVAL, "%s: bad argument", who);
    GreenUser u{G, mem};
    int rc = for_chunks(c, sites, n_sites, proposals, mem, who, [](gfmc_ctx* c, int first, int P, void* user) {
        auto* u = static_cast<GreenUser*>(user);
        const size_t per = (size_t)c->K * 4 * 16;
        for (int s0 = 0; s0 < P; s0 += c->lay.g_chunk) {
            const int n = std::min(c->lay.g_chunk, P - s0);
            int rc = run_green(c, s0, n, c->ptr<double2>(c->lay.Gbuf), nullptr, 0, nullptr);
            if (rc) return rc;
            rc = copy_out(c, reinterpret_cast<char*>(u->G) + (size_t)(first + s0) * per, c->ptr<char>(c->lay.Gbuf), (size_t)n * per, u->mem);
            if (rc) return rc;
        }
        return (int)GFMC_OK;
    }, &u);
    if (rc) return rc;
    return guard.finish();
}

int gfmc_local_green(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, double* E, double* G, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_local_green");
    if (c->mode == kModeDex && G) return fail(c, GFMC_EINVAL, "gfmc_local_green: model is GFMC_MODEL_DEX_INF, use gfmc_local_green_ov");
    return green_impl(c, guard, sites, n_sites, nullptr, E, G, mem, "gfmc_local_green");
}

int gfmc_local_green_ov(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, double* E, double* G, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_local_green_ov");
    if (c->mode != kModeDex) return fail(c, GFMC_EINVAL, "gfmc_local_green_ov: model is GFMC_MODEL_HUND, use gfmc_local_green");
    if (G && !proposals) return fail(c, GFMC_EINVAL, "gfmc_local_green_ov: NULL proposals");
    return green_impl(c, guard, sites, n_sites, proposals, E, G, mem, "gfmc_local_green_ov");
}

int gfmc_hopping(gfmc_ctx* c, double* Tb, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_hopping");
    if (!Tb || (mem != GFMC_HOST && mem != GFMC_DEVICE)) return fail(c, GFMC_EINVAL, "gfmc_hopping: bad argument");
    if (c->mode != kModeDex) return fail(c, GFMC_EINVAL, "gfmc_hopping: model is not GFMC_MODEL_DEX_INF");
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "gfmc_hopping: spins not set");
    CU_TRY(c, cudaSetDevice(c->p.device));
    const size_t nb = (size_t)16 * c->N;
    char* out = reinterpret_cast<char*>(Tb);
    int rc = copy_out(c, out, c->ptr<char>(c->lay.Tx), nb, mem); if (rc) return rc;
    rc = copy_out(c, out + nb, c->ptr<char>(c->lay.Ty), nb, mem); if (rc) return rc;
    rc = copy_out(c, out + 2 * nb, c->ptr<char>(c->lay.Tz), nb, mem); if (rc) return rc;
    return guard.finish();
}

struct DSUser { const double* prop; double* dS; int mem; };
int gfmc_delta_S(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, double* dS, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_delta_S");
    if (!proposals || !dS) return fail(c, GFMC_EINVAL, "gfmc_delta_S: NULL argument");
    DSUser u{proposals, dS, mem};
    int rc = for_chunks(c, sites, n_sites, proposals, mem, "gfmc_delta_S", [](gfmc_ctx* c, int first, int P, void* user) {
        auto* u = static_cast<DSUser*>(user);
        int rc = run_green(c, 0, P, nullptr, c->ptr<double>(c->lay.prop), 0, c->ptr<double>(c->lay.dS));
        if (rc) return rc;
        return copy_out(c, u->dS + first, c->ptr<double>(c->lay.dS), (size_t)P * 8, u->mem);
    }, &u);
    if (rc) return rc;
    return guard.finish();
}

// one frozen-batch update for the P sites in ctx->sites; proposals/uniforms already on the device.
static int update_batch_device(gfmc_ctx* c, int P, const double* prop_dev, const double* uni_dev, int by_site,
                               uint8_t* accepted_dev, double* dS_log_dev, uint8_t* acc_log_dev, unsigned long long* counter_dev, int apply = 1)
{
    if (c->batch_mode == GFMC_BATCH_EXACT && !apply)
        return fail(c, GFMC_EINVAL, "gfmc_decide_batch: decisions of an exact batch depend on each other; only GFMC_BATCH_FROZEN can be sharded");
    if (c->batch_mode == GFMC_BATCH_EXACT)
        return run_exact_batch(c, P, prop_dev, uni_dev, by_site, accepted_dev, dS_log_dev, acc_log_dev, counter_dev);
    int rc = run_moments_batch(c, P, prop_dev, by_site);
    if (rc) return rc;
    rc = run_green(c, 0, P, nullptr, prop_dev, by_site, c->ptr<double>(c->lay.dS));
    if (rc) return rc;
    MetropolisArgs ma{};
    ma.sites = c->ptr<int32_t>(c->lay.sites); ma.dS = c->ptr<double>(c->lay.dS);
    ma.proposals = prop_dev; ma.uniforms = uni_dev;
    ma.Sx = c->ptr<double>(c->lay.Sx); ma.Sy = c->ptr<double>(c->lay.Sy); ma.Sz = c->ptr<double>(c->lay.Sz);
    ma.accepted = accepted_dev; ma.dS_log = dS_log_dev; ma.accept_log = acc_log_dev; ma.n_accepted = counter_dev;
    ma.n = P; ma.by_site = by_site; ma.apply = apply;
    metropolis_kernel<<<(P + 255) / 256, 256, 0, c->stream>>>(ma);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return apply ? refresh_bonds(c) : GFMC_OK;          // "update H" (Alg. 1 line 12): the bond amplitudes follow the accepted flips
}

static int batch_entry(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, const double* uniforms,
                       double* dS, uint8_t* accepted, int mem, int apply)
{
    if (!c) return GFMC_EINVAL;
    const char* who = apply ? "gfmc_update_batch" : "gfmc_decide_batch";
    CallGuard guard(c, who);
    if (!sites || !proposals || !uniforms || n_sites < 0 || (mem != GFMC_HOST && mem != GFMC_DEVICE))
        return fail(c, GFMC_EINVAL, "%s: bad argument", who);
    if (n_sites > c->p.max_batch_sites) return fail(c, GFMC_EINVAL, "%s: n_sites %d > max_batch_sites %d", who, n_sites, c->p.max_batch_sites);
    if (c->batch_mode == GFMC_BATCH_EXACT && n_sites > c->p.exact_batch_sites)
        return fail(c, GFMC_EINVAL, "%s: n_sites %d > exact_batch_sites %d in GFMC_BATCH_EXACT mode", who, n_sites, c->p.exact_batch_sites);
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "%s: spins not set", who);
    if (n_sites == 0) return GFMC_OK;
    CU_TRY(c, cudaSetDevice(c->p.device));
    if (mem == GFMC_HOST) {
        int rc = check_sites_host(c, sites, n_sites); if (rc) return rc;
        std::vector<int32_t> tmp(sites, sites + n_sites);
        std::sort(tmp.begin(), tmp.end());
        if (std::adjacent_find(tmp.begin(), tmp.end()) != tmp.end()) return fail(c, GFMC_EINVAL, "%s: sites must be distinct", who);
        for (int i = 0; i < n_sites; ++i)
            if (!(uniforms[i] > 0.0 && uniforms[i] <= 1.0)) return fail(c, GFMC_EINVAL, "%s: uniforms must lie in (0,1]", who);
    }
    int rc = copy_in(c, c->ptr<int32_t>(c->lay.sites), sites, (size_t)n_sites * 4, mem); if (rc) return rc;
    rc = copy_in(c, c->ptr<double>(c->lay.prop), proposals, (size_t)n_sites * 24, mem); if (rc) return rc;
    rc = copy_in(c, c->ptr<double>(c->lay.uni), uniforms, (size_t)n_sites * 8, mem); if (rc) return rc;
    unsigned long long* counter = c->ptr<unsigned long long>(c->lay.scal) + 8;
    CU_TRY(c, cudaMemsetAsync(counter, 0, 8, c->stream));
    rc = update_batch_device(c, n_sites, c->ptr<double>(c->lay.prop), c->ptr<double>(c->lay.uni), 0,
                             c->ptr<uint8_t>(c->lay.acc), nullptr, nullptr, counter, apply);
    if (rc) return rc;
    if (dS) { rc = copy_out(c, dS, c->ptr<double>(c->lay.dS), (size_t)n_sites * 8, mem); if (rc) return rc; }
    if (accepted) { rc = copy_out(c, accepted, c->ptr<uint8_t>(c->lay.acc), (size_t)n_sites, mem); if (rc) return rc; }
    return guard.finish();
}

int gfmc_update_batch(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, const double* uniforms,
                      double* dS, uint8_t* accepted, int mem)
{
    return batch_entry(c, sites, n_sites, proposals, uniforms, dS, accepted, mem, 1);
}

// the two halves of a frozen-batch update, for one chain whose batches are sharded over several GPUs.  Every rank
// holds the whole spin field, decides its share of the batch against it (gfmc_decide_batch: a2-a6 + the accept test, configuration
// untouched), the ranks exchange (accepted, dS) with one all-gather, and every rank applies ALL accepted flips (gfmc_apply_flips).
int gfmc_decide_batch(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, const double* uniforms,
                      double* dS, uint8_t* accepted, int mem)
{
    return batch_entry(c, sites, n_sites, proposals, uniforms, dS, accepted, mem, 0);
}

int gfmc_apply_flips(gfmc_ctx* c, const int32_t* sites, int32_t n_sites, const double* proposals, const uint8_t* accepted, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_apply_flips");
    if (!sites || !proposals || !accepted || n_sites < 0 || (mem != GFMC_HOST && mem != GFMC_DEVICE))
        return fail(c, GFMC_EINVAL, "gfmc_apply_flips: bad argument");
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "gfmc_apply_flips: spins not set");
    if (n_sites == 0) return GFMC_OK;
    CU_TRY(c, cudaSetDevice(c->p.device));
    if (mem == GFMC_HOST) {
        // this is where the shares of a sharded batch meet: a wrong cut shows up here as a repeated site, which would make the
        // flips race and count twice.  Host lists are checked; device lists are trusted, as everywhere in this API.
        int rc = check_sites_host(c, sites, n_sites); if (rc) return rc;
        std::vector<int32_t> tmp(sites, sites + n_sites);
        std::sort(tmp.begin(), tmp.end());
        if (std::adjacent_find(tmp.begin(), tmp.end()) != tmp.end()) return fail(c, GFMC_EINVAL, "gfmc_apply_flips: sites must be distinct");
    }
    // staged in chunks of max_batch_sites through the context's buffers (the list may be a whole sharded batch: G x max_batch_sites)
    unsigned long long* counter = c->ptr<unsigned long long>(c->lay.scal) + 8;
    CU_TRY(c, cudaMemsetAsync(counter, 0, 8, c->stream));
    const int B = c->p.max_batch_sites;
    for (int first = 0; first < n_sites; first += B) {
        const int P = std::min(B, n_sites - first);
        int rc = copy_in(c, c->ptr<int32_t>(c->lay.sites), sites + first, (size_t)P * 4, mem); if (rc) return rc;
        rc = copy_in(c, c->ptr<double>(c->lay.prop), proposals + (size_t)first * 3, (size_t)P * 24, mem); if (rc) return rc;
        rc = copy_in(c, c->ptr<uint8_t>(c->lay.acc), accepted + first, (size_t)P, mem); if (rc) return rc;
        apply_flips_kernel<<<(P + 255) / 256, 256, 0, c->stream>>>(c->ptr<int32_t>(c->lay.sites), c->ptr<double>(c->lay.prop), c->ptr<uint8_t>(c->lay.acc), P,
                                                                  c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy), c->ptr<double>(c->lay.Sz), counter);
        c->counts[1] += 1;
        CU_TRY(c, cudaGetLastError());
    }
    int rc = refresh_bonds(c); if (rc) return rc;
    return guard.finish();
}

// One frozen-batch update of a sweep as a replayed CUDA graph (see sweep_device).  The graph is keyed by what is baked into its
// nodes: P, the temperature and which logs are written.  The trial moves and the logs of a graph-replayed sweep always live in
// the context's own staging buffers (gfmc_sweep copies device-resident caller arrays there, N x 32 bytes per sweep), so the
// pointers never change from sweep to sweep and a graph is captured once per (P, T); the batch cursor and the acceptance
// counter live on the device.  The cache is a small LRU: an evicted graph is destroyed only after the stream has drained.
static int launch_batch_graph(gfmc_ctx* c, int P, const double* prop_dev, const double* uni_dev, double* dlog_dev, uint8_t* alog_dev,
                              unsigned long long* counter, int* cursor)
{
    for (auto& gr : c->graphs)
        if (gr.P == P && gr.prop == prop_dev && gr.uni == uni_dev && gr.dlog == dlog_dev && gr.alog == alog_dev && gr.T == c->p.T) {
            CU_TRY(c, cudaGraphLaunch(gr.exec, c->stream));
            gr.used = ++c->graph_clock;
            c->counts[0] += gr.n0; c->counts[1] += gr.n1;
            return GFMC_OK;
        }
    if (c->graphs.size() >= 8) {
        size_t lru = 0;
        for (size_t k = 1; k < c->graphs.size(); ++k) if (c->graphs[k].used < c->graphs[lru].used) lru = k;
        CU_TRY(c, cudaStreamSynchronize(c->stream));          // the evicted graph may still be in flight
        cudaGraphExecDestroy(c->graphs[lru].exec);
        c->graphs.erase(c->graphs.begin() + (long)lru);
    }
    const int64_t n0 = c->counts[0], n1 = c->counts[1];
    cudaGraph_t graph = nullptr;
    CU_TRY(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    c->capturing = true;
    next_batch_kernel<<<1, 1024, 0, c->stream>>>(c->ptr<int32_t>(c->lay.order), cursor, c->ptr<int32_t>(c->lay.sites), P);
    c->counts[1] += 1;
    int rc = update_batch_device(c, P, prop_dev, uni_dev, 1, nullptr, dlog_dev, alog_dev, counter);
    c->capturing = false;
    cudaError_t ce = cudaStreamEndCapture(c->stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (ce != cudaSuccess) return fail(c, GFMC_ECUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(ce));
    gfmc_ctx::BatchGraph gr{P, prop_dev, uni_dev, dlog_dev, alog_dev, c->p.T, nullptr, c->counts[0] - n0, c->counts[1] - n1, ++c->graph_clock};
    ce = cudaGraphInstantiate(&gr.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ce != cudaSuccess) return fail(c, GFMC_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(ce));
    c->graphs.push_back(gr);
    CU_TRY(c, cudaGraphLaunch(gr.exec, c->stream));      // the capture did not execute anything: this is the batch itself
    return GFMC_OK;
}

// Does a sweep with this batch size replay CUDA graphs?  Launch-bound regime only: vectors resident in shared memory and many
// small batches per sweep.
static bool sweep_uses_graph(const gfmc_ctx* c, int batch_sites)
{
    const int nbatches = (c->ncolour[0] + batch_sites - 1) / batch_sites + (c->ncolour[1] + batch_sites - 1) / batch_sites;
    return !c->tun.no_graph && c->batch_mode == GFMC_BATCH_FROZEN && nbatches >= 8 && make_resident_plan(c->p.L, c->smem_limit, c->tun).ok;
}

// The two-colour schedule (x+y+z) mod 2 is a proper colouring of the periodic lattice only for even L: at odd L the wrap
// neighbours x = 0 and x = L-1 share a colour.  In the J_H->inf model two neighbouring flips change the SAME bond, so a frozen
// batch holding both would be wrong at first order in that bond (not at second order in G, as for sites that are not
// neighbours): refused.  batch_sites = 1 (the paper's sequential algorithm) is exact on any lattice.
static int check_schedule(gfmc_ctx* c, int batch_sites, const char* who)
{
    if (c->batch_mode == GFMC_BATCH_EXACT && batch_sites > c->p.exact_batch_sites)
        return fail(c, GFMC_EINVAL, "%s: batch_sites %d > exact_batch_sites %d in GFMC_BATCH_EXACT mode", who, batch_sites, c->p.exact_batch_sites);
    if (c->mode == kModeDex && (c->p.L & 1) && batch_sites > 1)
        return fail(c, GFMC_EINVAL, "%s: odd L = %d with batch_sites > 1 puts nearest neighbours into one frozen batch of the J_H->inf model "
                                    "(they share a bond); use batch_sites = 1 or an even L", who, c->p.L);
    return GFMC_OK;
}

// One sweep (both colours, consecutive batches of batch_sites) with device-resident trial spins / uniforms indexed by site;
// leaves the magnetization in scal[0] and the number of accepted flips in the counter behind it.  run_stats: see magnetization_kernel.
static int sweep_device(gfmc_ctx* c, int batch_sites, const double* prop_dev, const double* uni_dev, double* dlog_dev, uint8_t* alog_dev,
                        double* run_stats)
{
    double* scal = c->ptr<double>(c->lay.scal);
    unsigned long long* counter = c->ptr<unsigned long long>(c->lay.scal) + 8;
    CU_TRY(c, cudaMemsetAsync(counter, 0, 8, c->stream));
    // Launch-bound regime (vectors resident in shared memory, many small batches per sweep): the per-batch sequence
    // (gather sites -> a2/a3 -> moments -> a4-a6 -> a7 [-> bond refresh]) has constant arguments once the batch cursor lives on the
    // device, so it is captured once as a CUDA graph and replayed for every batch of the sweep.
    const bool use_graph = sweep_uses_graph(c, batch_sites);
    int* cursor = reinterpret_cast<int*>(c->ptr<unsigned long long>(c->lay.scal) + 16);
    if (use_graph) CU_TRY(c, cudaMemsetAsync(cursor, 0, 4, c->stream));
    int base = 0;
    for (int col = 0; col < 2; ++col) {
        for (int st = 0; st < c->ncolour[col]; st += batch_sites) {
            const int P = std::min(batch_sites, c->ncolour[col] - st);
            if (use_graph) {
                int rc = launch_batch_graph(c, P, prop_dev, uni_dev, dlog_dev, alog_dev, counter, cursor);
                if (rc) return rc;
            } else {
                CU_TRY(c, cudaMemcpyAsync(c->ptr<int32_t>(c->lay.sites), c->ptr<int32_t>(c->lay.order) + base + st, (size_t)P * 4,
                                          cudaMemcpyDeviceToDevice, c->stream));
                int rc = update_batch_device(c, P, prop_dev, uni_dev, 1, nullptr, dlog_dev, alog_dev, counter);
                if (rc) return rc;
            }
            // Keep at most 2 x 32 batches queued.  A host thread that runs thousands of launches ahead ends up blocked inside
            // the driver on a full queue, and while it waits there the launches of other contexts' threads wait with it
            // (measured: 8 concurrent chains slower than 4 without this).
            if (++c->throttle_n % 32 == 0) {
                const int k = (int)((c->throttle_n / 32) & 1);
                if (!c->throttle_ev[k]) CU_TRY(c, cudaEventCreateWithFlags(&c->throttle_ev[k], cudaEventDisableTiming | cudaEventBlockingSync));   // sleep, do not spin: more chains than host cores
                else CU_TRY(c, cudaEventSynchronize(c->throttle_ev[k]));
                CU_TRY(c, cudaEventRecord(c->throttle_ev[k], c->stream));
            }
        }
        base += c->ncolour[col];
    }
    magnetization_kernel<<<1, 1024, 0, c->stream>>>(c->ptr<double>(c->lay.Sx), c->ptr<double>(c->lay.Sy), c->ptr<double>(c->lay.Sz), c->N, scal,
                                                    run_stats, counter);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    return GFMC_OK;
}

int gfmc_sweep(gfmc_ctx* c, int32_t n_sweeps, int32_t batch_sites, const double* proposals, const double* uniforms,
               double* dS_log, uint8_t* accept_log, double* magnetization, int64_t* n_accepted, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_sweep");
    if (!proposals || !uniforms || n_sweeps < 0 || batch_sites < 1 || (mem != GFMC_HOST && mem != GFMC_DEVICE))
        return fail(c, GFMC_EINVAL, "gfmc_sweep: bad argument");
    if (batch_sites > c->p.max_batch_sites) return fail(c, GFMC_EINVAL, "gfmc_sweep: batch_sites %d > max_batch_sites %d", batch_sites, c->p.max_batch_sites);
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "gfmc_sweep: spins not set");
    { int rc = check_schedule(c, batch_sites, "gfmc_sweep"); if (rc) return rc; }
    CU_TRY(c, cudaSetDevice(c->p.device));
    const size_t N = c->N;
    double* scal = c->ptr<double>(c->lay.scal);
    unsigned long long* counter = c->ptr<unsigned long long>(c->lay.scal) + 8;
    // graph-replayed sweeps read their trial moves from, and write their logs to, the context's staging buffers whatever `mem` is
    const bool stage = (mem == GFMC_HOST) || sweep_uses_graph(c, batch_sites);
    for (int s = 0; s < n_sweeps; ++s) {
        const double* prop_s = proposals + (size_t)s * N * 3;
        const double* uni_s = uniforms + (size_t)s * N;
        const double* prop_dev; const double* uni_dev;
        double* dlog_dev = nullptr; uint8_t* alog_dev = nullptr;
        if (stage) {
            if (mem == GFMC_HOST)
                for (size_t i = 0; i < N; ++i)
                    if (!(uni_s[i] > 0.0 && uni_s[i] <= 1.0)) return fail(c, GFMC_EINVAL, "gfmc_sweep: uniforms must lie in (0,1]");
            int rc = copy_in(c, c->ptr<double>(c->lay.prop), prop_s, N * 24, mem); if (rc) return rc;
            rc = copy_in(c, c->ptr<double>(c->lay.uni), uni_s, N * 8, mem); if (rc) return rc;
            prop_dev = c->ptr<double>(c->lay.prop); uni_dev = c->ptr<double>(c->lay.uni);
            if (dS_log) dlog_dev = c->ptr<double>(c->lay.logdS);
            if (accept_log) alog_dev = c->ptr<uint8_t>(c->lay.logacc);
        } else {
            prop_dev = prop_s; uni_dev = uni_s;
            if (dS_log) dlog_dev = dS_log + (size_t)s * N;
            if (accept_log) alog_dev = accept_log + (size_t)s * N;
        }
        { int rc = sweep_device(c, batch_sites, prop_dev, uni_dev, dlog_dev, alog_dev, nullptr); if (rc) return rc; }
        if (magnetization) { int rc = copy_out(c, magnetization + s, scal, 8, mem); if (rc) return rc; }
        if (n_accepted) { int rc = copy_out(c, n_accepted + s, counter, 8, mem); if (rc) return rc; }
        if (stage) {
            if (dS_log) { int rc = copy_out(c, dS_log + (size_t)s * N, dlog_dev, N * 8, mem); if (rc) return rc; }
            if (accept_log) { int rc = copy_out(c, accept_log + (size_t)s * N, alog_dev, N, mem); if (rc) return rc; }
            // host memory: the staging buffers are reused by the next sweep, finish the copies first (device copies are stream-ordered)
            if (mem == GFMC_HOST) CU_TRY(c, cudaStreamSynchronize(c->stream));
        }
    }
    return guard.finish();
}

// f5: how the sites of one batch are decided (gfmc_update_batch, gfmc_sweep, gfmc_run)
int gfmc_set_batch_mode(gfmc_ctx* c, int mode)
{
    if (!c) return GFMC_EINVAL;
    c->err.clear();
    if (mode != GFMC_BATCH_FROZEN && mode != GFMC_BATCH_EXACT) return fail(c, GFMC_EINVAL, "gfmc_set_batch_mode: unknown mode %d", mode);
    if (mode == GFMC_BATCH_EXACT && c->p.exact_batch_sites <= 0)
        return fail(c, GFMC_ESTATE, "gfmc_set_batch_mode: the context was created with exact_batch_sites = 0");
    c->batch_mode = mode;
    return GFMC_OK;
}

// f3: temperature of the chain (the only place T enters is beta in the Delta S_eff quadrature, Eq. (14)): lets one context
// anneal through a temperature list, as the M(T) curves of the paper's validation do (Fig. 4).
int gfmc_set_temperature(gfmc_ctx* c, double T)
{
    if (!c) return GFMC_EINVAL;
    c->err.clear();
    if (!(T > 0.0) || !std::isfinite(T)) return fail(c, GFMC_EINVAL, "gfmc_set_temperature: T must be positive and finite");
    c->p.T = T;
    return GFMC_OK;
}

// f3: the trial moves of Algorithm 1 from the library's own counter-based generator (post.cuh, reading f3-1).
int gfmc_random_proposals(gfmc_ctx* c, uint64_t seed, int64_t sweep, double* proposals, double* uniforms, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_random_proposals");
    if (!proposals || !uniforms || sweep < 0 || (mem != GFMC_HOST && mem != GFMC_DEVICE)) return fail(c, GFMC_EINVAL, "gfmc_random_proposals: bad argument");
    CU_TRY(c, cudaSetDevice(c->p.device));
    const size_t N = c->N;
    double* pd = (mem == GFMC_DEVICE) ? proposals : c->ptr<double>(c->lay.prop);
    double* ud = (mem == GFMC_DEVICE) ? uniforms : c->ptr<double>(c->lay.uni);
    propose_kernel<<<(unsigned)((N + 255) / 256), 256, 0, c->stream>>>(seed, (unsigned long long)sweep, (int)N, pd, ud);
    c->counts[1] += 1;
    CU_TRY(c, cudaGetLastError());
    if (mem == GFMC_HOST) {
        int rc = copy_out(c, proposals, pd, N * 24, mem); if (rc) return rc;
        rc = copy_out(c, uniforms, ud, N * 8, mem); if (rc) return rc;
    }
    return guard.finish();
}

// f3: Algorithm 1 end to end on the device: sweeps first_sweep .. first_sweep + n_sweeps - 1 of the chain `seed`,
// trial moves drawn on the device, nothing but the per-sweep observables crosses the bus.
int gfmc_run(gfmc_ctx* c, uint64_t seed, int64_t first_sweep, int32_t n_sweeps, int32_t batch_sites,
             double* magnetization, int64_t* n_accepted, int mem)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_run");
    if (first_sweep < 0 || n_sweeps < 0 || batch_sites < 1 || (mem != GFMC_HOST && mem != GFMC_DEVICE)) return fail(c, GFMC_EINVAL, "gfmc_run: bad argument");
    if (batch_sites > c->p.max_batch_sites) return fail(c, GFMC_EINVAL, "gfmc_run: batch_sites %d > max_batch_sites %d", batch_sites, c->p.max_batch_sites);
    if (!c->spins_set) return fail(c, GFMC_ESTATE, "gfmc_run: spins not set");
    { int rc = check_schedule(c, batch_sites, "gfmc_run"); if (rc) return rc; }
    CU_TRY(c, cudaSetDevice(c->p.device));
    const size_t N = c->N;
    double* scal = c->ptr<double>(c->lay.scal);
    unsigned long long* counter = c->ptr<unsigned long long>(c->lay.scal) + 8;
    double* run_stats = scal + 24;           // (S, mean m, sum of squared deviations, accepted flips) of this call: Alg. 1 lines 16-17
    CU_TRY(c, cudaMemsetAsync(run_stats, 0, 4 * sizeof(double), c->stream));
    c->run_sweeps = 0;
    double* pd = c->ptr<double>(c->lay.prop);
    double* ud = c->ptr<double>(c->lay.uni);
    for (int s = 0; s < n_sweeps; ++s) {
        propose_kernel<<<(unsigned)((N + 255) / 256), 256, 0, c->stream>>>(seed, (unsigned long long)(first_sweep + s), (int)N, pd, ud);
        c->counts[1] += 1;
        int rc = sweep_device(c, batch_sites, pd, ud, nullptr, nullptr, run_stats); if (rc) return rc;
        if (magnetization) { rc = copy_out(c, magnetization + s, scal, 8, mem); if (rc) return rc; }
        if (n_accepted) { rc = copy_out(c, n_accepted + s, counter, 8, mem); if (rc) return rc; }
    }
    int rc = guard.finish();
    if (rc == GFMC_OK) c->run_sweeps = n_sweeps;
    return rc;
}

// f3: Alg. 1 lines 16-17 ("return M/S") for the sweeps of the most recent gfmc_run call, from the running
// statistics that magnetization_kernel keeps on the device.
int gfmc_run_summary(gfmc_ctx* c, double* mean_magnetization, double* stderr_magnetization, double* acceptance, int64_t* n_sweeps)
{
    if (!c) return GFMC_EINVAL;
    CallGuard guard(c, "gfmc_run_summary");
    if (c->run_sweeps <= 0) return fail(c, GFMC_ESTATE, "gfmc_run_summary: no completed gfmc_run with n_sweeps > 0 on this context");
    CU_TRY(c, cudaSetDevice(c->p.device));
    double st[4];
    CU_TRY(c, cudaMemcpyAsync(st, c->ptr<double>(c->lay.scal) + 24, sizeof st, cudaMemcpyDeviceToHost, c->stream));
    int rc = guard.finish(); if (rc) return rc;
    if (mean_magnetization) *mean_magnetization = st[1];
    if (stderr_magnetization) *stderr_magnetization = st[0] > 1.0 ? std::sqrt(st[2] / (st[0] - 1.0) / st[0]) : std::nan("");
    if (acceptance) *acceptance = st[3] / (st[0] * (double)c->N);
    if (n_sweeps) *n_sweeps = (int64_t)st[0];
    return GFMC_OK;
}

}  // extern "C"

// ------------------------------------------------------------------ gfmc_moments_static: the entry point that allocates nothing
//
// Who needs it.  Some programs that link this library are not allowed to ask CUDA for device memory at the moment they want
// moments: a trainer or server that gave the whole GPU to its own pool allocator at start-up (a later cudaMalloc simply returns
// out-of-memory, or fragments the pool's view of the device); a thread working next to another thread's global-mode stream
// capture, which an allocation call would invalidate; a real-time loop that cannot take the device-wide synchronisation a
// cudaMalloc / cudaFree pair implies.  gfmc_create sizes and allocates (or adopts) a workspace, so those callers cannot get past
// it.  This entry point needs no context: the scratch memory of the shared-memory-resident path -- the SoA copy of the spin
// field and the per-step Gram sums that cheb_resident_kernel hands to finalize_moments -- lives in the fixed array below, which is
// part of the library image (every device that loads libgfmc.so carries these 4.05 MiB until the process exits).
//
// The array is shared by every call on a device and keeps the previous call's contents.  Nothing in it has to start at zero:
// spins_aos_to_soa overwrites Sx, Sy, Sz for all N sites and the resident kernel writes every Gram entry (step, site, k) that
// finalize_moments reads, so no clearing pass is needed.  Two calls that overlap on one GPU (two host threads, or two streams)
// would write the same bytes: they race, and the caller has to serialise them.
namespace {

constexpr int    kStaticMaxL         = 12;                      // the resident kernel's limit (128 L^3 bytes of shared memory)
constexpr size_t kStaticSpinStride   = 2048;                    // >= 12^3 = 1728 doubles per spin component
constexpr size_t kStaticMaxStepSites = GFMC_STATIC_MAX_STEP_SITES;      // (M/2) * n_sites
constexpr size_t kStaticGramDoubles  = kStaticMaxStepSites * 8; // gram_width(kModeHund2) = 8 sums per (step, site)
constexpr size_t kStaticDoubles      = 3 * kStaticSpinStride + kStaticGramDoubles;

// Host code may not use this name as a pointer (on the host it is only a handle for cudaGetSymbolAddress); kernels get the
// device address looked up in static_setup().
static __device__ __align__(256) double g_static_scratch[kStaticDoubles];

struct StaticDevice { bool ready; double* scratch; int smem_limit; };
constexpr int kStaticMaxDevices = 64;
StaticDevice g_static_dev[kStaticMaxDevices];        // zero-initialised; guarded by g_static_mutex
std::mutex g_static_mutex;
thread_local char g_static_error[320];

int static_fail(int code, const char* fmt, ...)
{
    va_list ap; va_start(ap, fmt); vsnprintf(g_static_error, sizeof g_static_error, fmt, ap); va_end(ap);
    return code;
}

#define CU_TRY_STATIC(expr)                                                                         \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return static_fail(GFMC_ECUDA, "gfmc_moments_static: %s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

// Once per device, with that device current: the device address of the scratch array, and the opt-in to large dynamic shared
// memory for the four instances of the resident kernel this entry point launches.  No allocation call.
int static_setup(int device, StaticDevice* out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& d = g_static_dev[device];
    if (!d.ready) {
        int major = 0, smem = 0;
        CU_TRY_STATIC(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
        if (major != 10) return static_fail(GFMC_ECUDA, "gfmc_moments_static: device %d is sm_%dx; libgfmc is built for sm_100a only", device, major);
        CU_TRY_STATIC(cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
        double* ptr = nullptr;
        CU_TRY_STATIC(cudaGetSymbolAddress((void**)&ptr, g_static_scratch));
        if (!ptr) return static_fail(GFMC_ECUDA, "gfmc_moments_static: cudaGetSymbolAddress returned a null address");
        CU_TRY_STATIC(set_resident_smem_limit_mode<kModeHund2>(smem));
        d.scratch = ptr; d.smem_limit = smem; d.ready = true;
    }
    *out = d;
    return GFMC_OK;
}

struct DeviceRestore {          // leaves the calling thread's current device as it found it
    int prev = -1;
    ~DeviceRestore() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

extern "C" {

const char* gfmc_moments_static_error(void) { return g_static_error; }

int gfmc_moments_static(int32_t device, void* stream, int32_t L, int32_t M, double t, double JH,
                        const double* S, const int32_t* sites, int32_t n_sites, double* mu)
{
    nvtxRangePushA("gfmc_moments_static");
    struct Pop { ~Pop() { nvtxRangePop(); } } pop;
    g_static_error[0] = 0;
    if (L < 2 || L > kStaticMaxL)
        return static_fail(GFMC_EINVAL, "gfmc_moments_static: L = %d outside 2..%d (larger lattices do not fit the shared-memory-resident kernel; "
                                        "use gfmc_create + gfmc_moments)", L, kStaticMaxL);
    if (M < 2 || (M & 1)) return static_fail(GFMC_EINVAL, "gfmc_moments_static: M = %d must be even and >= 2", M);
    if (n_sites < 0) return static_fail(GFMC_EINVAL, "gfmc_moments_static: n_sites = %d is negative", n_sites);
    if ((size_t)(M / 2) * (size_t)n_sites > kStaticMaxStepSites)
        return static_fail(GFMC_EINVAL, "gfmc_moments_static: (M/2) * n_sites = %zu exceeds the fixed scratch array's maximum of %zu "
                                        "(GFMC_STATIC_MAX_STEP_SITES); split the site list or use gfmc_create + gfmc_moments",
                           (size_t)(M / 2) * (size_t)n_sites, kStaticMaxStepSites);
    if (!std::isfinite(t) || !std::isfinite(JH) || (t == 0.0 && JH == 0.0))
        return static_fail(GFMC_EINVAL, "gfmc_moments_static: t and J_H must be finite and not both zero");
    if (n_sites == 0) return GFMC_OK;
    if (!S || !sites || !mu) return static_fail(GFMC_EINVAL, "gfmc_moments_static: NULL pointer");
    if (device < 0 || device >= kStaticMaxDevices) return static_fail(GFMC_EINVAL, "gfmc_moments_static: device %d outside 0..%d", device, kStaticMaxDevices - 1);
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        (void)cudaGetLastError();
        return static_fail(GFMC_ECUDA, "gfmc_moments_static: no CUDA device: %s (libgfmc has no CPU fallback)",
                           e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    if (device >= ndev) return static_fail(GFMC_EINVAL, "gfmc_moments_static: device %d out of range (%d present)", device, ndev);

    DeviceRestore restore;
    int cur = -1;
    CU_TRY_STATIC(cudaGetDevice(&cur));
    if (cur != device) { CU_TRY_STATIC(cudaSetDevice(device)); restore.prev = cur; }
    StaticDevice dev{};
    if (int rc = static_setup(device, &dev)) return rc;

    const int N = L * L * L, P = n_sites;
    const ResidentPlan rp = make_resident_plan(L, (size_t)dev.smem_limit, Tuning{});
    if (!rp.ok) return static_fail(GFMC_ECUDA, "gfmc_moments_static: %zu bytes of shared memory per CTA needed, device offers %d", rp.smem_bytes, dev.smem_limit);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    double* Sx = dev.scratch;
    double* Sy = Sx + kStaticSpinStride;
    double* Sz = Sy + kStaticSpinStride;
    double* gram = Sz + kStaticSpinStride;

    const double a = 6.0 * std::fabs(t) + std::sqrt(2.0) * std::fabs(JH);        // a1, as gfmc_create
    spins_aos_to_soa<<<(N + 127) / 128, 128, 0, st>>>(S, Sx, Sy, Sz, N);
    ResidentArgs ra{};
    ra.sites = sites;
    ra.Sx = Sx; ra.Sy = Sy; ra.Sz = Sz;
    ra.gram = gram;
    ra.t_over_a = t / a; ra.jh_over_a = JH / a;
    ra.L = L; ra.N = N; ra.Npad = rp.Npad; ra.G = rp.G; ra.P = P; ra.Ps = P; ra.nsteps = M / 2;
    launch_resident_mode<kModeHund2>(rp.spt, (unsigned)((P + rp.G - 1) / rp.G), rp.smem_bytes, st, ra);
    const long long nthreads = (long long)P * (M / 2 + 1);
    finalize_moments<<<(unsigned)((nthreads + 255) / 256), 256, 0, st>>>(gram, reinterpret_cast<double2*>(mu), P, M, 1);
    e = cudaGetLastError();
    cudaError_t es = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = es;
    if (e != cudaSuccess) { (void)cudaGetLastError(); return static_fail(GFMC_ECUDA, "gfmc_moments_static: launch failed: %s", cudaGetErrorString(e)); }
    return GFMC_OK;
}

}  // extern "C"
