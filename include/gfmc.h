/*
 * gfmc.h -- C ABI of libgfmc.so: the data-parallel hot path of the O(N)
 * Green-function-based Monte Carlo (GFMC) method for the 3D double-exchange model
 * (arXiv:1303.6016), hand-written CUDA for NVIDIA B200 (sm_100a), fp64.
 *
 * Citations are lines of the paper text with the equation / algorithm they
 * fall in.  Where the paper is silent the reading is the one listed in DESIGN.md.
 *
 * What the library computes (one "site update", Algorithm 1 lines 3-13):
 *   H   = -t sum_<ij>,s (c+_is c_js + h.c.) + J_H sum_i S_i . c+_ia sigma_ab c_ib       Eq. (1)
 *   H~  = (H - b)/a,  a = 6|t| + sqrt(2)|J_H|, b = 0                                       rescaling
 *   |r_0> = |o s>, |r_1> = H~|r_0>, |r_m> = 2 H~|r_{m-1}> - |r_{m-2}>                       Eq. (26)
 *   mu_{2m-i}(a,b) = 2 <r^a_{m-i}|r^b_m> - mu_i(a,b), i = 0,1                               Eq. (27)-(28)
 *   G~_ab(x_k) = (2i/sin phi_k) sum_m mu'_m(a,b) e^{-i m phi_k}, phi_k = pi(k+1/2)/K        Eq. (24),(29)-(30)
 *   d(z) = Det[1 + G(z) Delta], Delta = H' - H = J_H (S'_o - S_o).sigma (2x2 on-site)       Eq. (11),(17)-(22)
 *   Delta S_eff = (beta/pi) Int f(E) Im log d(E + i0) dE                                    Eq. (14)
 *   accept iff exp(-Delta S_eff) > rand()                                                   Alg. 1 line 10
 *
 * Conventions
 *   - Lattice: periodic simple cubic, edge L >= 2, N = L^3 sites, site i = x + L*(y + L*z).
 *     Matrix dimension D = 2N, row = 2*i + s, s = 0 (up), 1 (down).
 *   - All floating point is IEEE fp64.  Complex values are interleaved (re, im) doubles.
 *   - `mem` arguments: GFMC_HOST (0) = every pointer of that call is a host pointer,
 *     GFMC_DEVICE (1) = every pointer is a device pointer on the context's device.
 *   - Ownership: the context owns only what it allocates.  Caller pointers stay caller-owned
 *     and are read/written only during the call.  Every call is synchronous on return
 *     (the context's stream is synchronised before returning) unless stated otherwise.
 *   - Errors: every function returns 0 (GFMC_OK) or a negative code; nothing aborts or throws.
 *     gfmc_last_error(ctx) returns a context-owned NUL-terminated string, valid until the next
 *     call on that context.  There is no CPU fallback: without a CUDA device gfmc_create fails
 *     with GFMC_ECUDA.
 *   - Not thread-safe per context; different contexts may be used from different threads.
 *   - Kernel selection is automatic and does not change any result beyond rounding order: lattices with L <= 12 run the
 *     whole recursion out of shared memory (one launch per batch), larger ones stream the vectors through TMA rings (one
 *     launch per Chebyshev step); the node sums of Eq. (24) use an FFT when n_energy is a power of two, the direct sum
 *     otherwise.  The library reads NO environment variable and keeps NO process-wide state: the diagnostic overrides used by
 *     the A/B measurements and the tests are per-context fields of gfmc_params (`flags`, `ring_stages_*`, `streamk_eff`).
 */
#ifndef GFMC_H
#define GFMC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GFMC_OK       0
#define GFMC_EINVAL  (-1)   /* bad argument: NULL, site out of range, M odd or < 2, batch > max_batch_sites, ... */
#define GFMC_ENOMEM  (-2)   /* device or host allocation failed / workspace too small */
#define GFMC_ECUDA   (-3)   /* a CUDA call failed; message in gfmc_last_error */
#define GFMC_ESTATE  (-4)   /* call out of order, e.g. spins not set */

#define GFMC_HOST    0
#define GFMC_DEVICE  1

#define GFMC_KERNEL_JACKSON 0   /* default (BASELINE.json) */
#define GFMC_KERNEL_LORENTZ 1   /* the paper's, g_m = sinh[lambda(1-m/M)]/sinh(lambda) */
#define GFMC_KERNEL_NONE    2

#define GFMC_MODEL_HUND     0   /* Eq. (1): finite J_H, dimension D = 2N (BASELINE.json's model; default) */
#define GFMC_MODEL_DEX_INF  1   /* Eq. (2)-(3): J_H -> infinity, dimension N, complex bond amplitudes t_ij --
                                   the Hamiltonian the paper's own runs use; J_H is ignored */

#define GFMC_FLAG_NO_RESIDENT   1   /* lattices with L <= 12 also run the streaming kernel (one launch per Chebyshev step) */
#define GFMC_FLAG_GREEN_DIRECT  2   /* node sums of Eq. (24) by the direct O(M K) sum even where the FFT kernel applies */
#define GFMC_FLAG_NO_GRAPH      4   /* sweeps launch every kernel individually instead of replaying one CUDA graph per batch */
#define GFMC_FLAG_NO_PDL       16   /* streaming step kernels are launched without programmatic dependent launch (each launch then starts only after
                                       the previous one has fully drained; the default overlaps a launch's start-up with the previous launch's tail) */
#define GFMC_FLAG_TWO_STEP      8   /* not a diagnostic: TWO Chebyshev steps per pass over the work vectors (temporal blocking):
                                       64 B instead of 96 B of HBM traffic per element and two steps, four work buffers instead of two.  Built for
                                       GFMC_MODEL_HUND with ph_symmetry = 1, L = 32 and M a multiple of 4 (GFMC_EINVAL otherwise).  Same moments to
                                       rounding order */

#define GFMC_BATCH_FROZEN  0   /* every site of a batch is evaluated against the configuration at batch start (default) */
#define GFMC_BATCH_EXACT   1   /* the sites of a batch are decided in order; each sees the earlier accepted flips of the batch exactly */

typedef struct gfmc_ctx gfmc_ctx;

typedef struct gfmc_params {
    int32_t L;                 /* lattice edge, 2 <= L <= 256 */
    int32_t M;                 /* number of Chebyshev moments, even, >= 2 ("Chebyshev truncation number") */
    int32_t n_energy;          /* K energy points of the Chebyshev-node grid; 0 -> 2*M */
    double  t;                 /* hopping */
    double  JH;                /* Hund coupling */
    double  T;                 /* temperature > 0 (beta = 1/T) */
    double  mu;                /* chemical potential (0 in the paper's runs) */
    int32_t kernel;            /* GFMC_KERNEL_* */
    double  lambda;            /* Lorentz kernel only; <= 0 -> 4 */
    int32_t max_batch_sites;   /* B_max: sizes the two work buffers, 2 * 16*D*2*B_max bytes */
    int32_t device;            /* CUDA device ordinal */
    void*   stream;            /* cudaStream_t the library launches on; NULL -> a context-owned stream; every call then first waits for
                                * the work already queued on the legacy default stream and synchronises before returning */
    void*   workspace;         /* optional caller-owned DEVICE memory (e.g. a torch tensor), 256-byte aligned */
    size_t  workspace_bytes;   /* must be >= gfmc_workspace_bytes(params) when workspace != NULL */
    int32_t model;             /* GFMC_MODEL_*; for GFMC_MODEL_DEX_INF: L >= 3, a = 6|t|, work buffers 16*N*2*B_max bytes each */
    int32_t ph_symmetry;       /* GFMC_MODEL_HUND, even L only.  1: propagate ONE start vector per site (|o up>) and obtain the
                                  Gram blocks of |o dn> from the antiunitary symmetry A = Gamma (i sigma_y) K, A H A^-1 = -H,
                                  of Eq. (1) on a bipartite periodic lattice: same moments to rounding,
                                  half the H-applications and half the work-buffer bytes per site.  0 (default): both start
                                  vectors are propagated, as rows a2-a3 of the scope table define the path. */
    /* Diagnostics, per context (0 = automatic everywhere; results are the same to rounding order whatever is set here): */
    int32_t flags;             /* bit mask of GFMC_FLAG_* */
    int32_t ring_stages_cur;   /* depth of the streaming kernel's R_cur ring (>= 3); 0 = as deep as shared memory allows */
    int32_t ring_stages_prev;  /* depth of its CTA-wide R_prev ring (>= 1; run-time-L kernel only: the per-warp rings of L = 8, 16, 32, 64 are one
                                  stage deep at compile time); 0 = automatic */
    double  streamk_eff;       /* mid-size batches walk a balanced explicit work list when whole-column work items would keep the SMs
                                  busy for less than this fraction of a launch; 0 -> 0.97 (default), < 0 -> never */
    int32_t exact_batch_sites; /* largest batch that may be decided exactly (GFMC_BATCH_EXACT, see gfmc_set_batch_mode): 0 (default) =
                                  not available; 1..64, <= max_batch_sites, GFMC_MODEL_HUND with ph_symmetry = 0 only.  Sizes two
                                  extra buffers of 64*(M + K)*exact_batch_sites^2 bytes. */
} gfmc_params;

/* Bytes of device memory a context with these parameters needs (0 on invalid parameters). */
size_t gfmc_workspace_bytes(const gfmc_params* params);

/* Creates a context (validates parameters, allocates or adopts the workspace, builds tables).
 * *out is NULL on failure; the error code tells why.  A failed create leaves no message behind;
 * gfmc_create_error() returns the text of the last failed create of the calling thread. */
int gfmc_create(const gfmc_params* params, gfmc_ctx** out);
const char* gfmc_create_error(void);
int gfmc_destroy(gfmc_ctx* ctx);                /* NULL is allowed */

/* Classical spins S [N][3] (site-major xyz), |S_i| = 1.  Copied into the context.
 * Host input is validated (| |S_i| - 1 | <= 1e-12, else GFMC_EINVAL); device input is trusted. */
int gfmc_set_spins(gfmc_ctx* ctx, const double* S, int mem);
int gfmc_get_spins(gfmc_ctx* ctx, double* S, int mem);

/* Spectral rescaling H~ = (H - b)/a (a1): a = 6|t| + sqrt(2)|J_H| (spin-independent Gershgorin bound), b = 0. */
int gfmc_bounds(const gfmc_ctx* ctx, double* a, double* b);

/* Undamped moments for n_sites sites (any order, repeats allowed; processed in chunks of max_batch_sites):
 *   mu[s][n][alpha][beta][re,im] = <o_s alpha| T_n(H~) |o_s beta>,  n = 0..M-1        Eq. (25)
 * computed with M/2 fused stencil+Chebyshev steps and the doubling of Eq. (27)-(28). */
int gfmc_moments(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites, double* mu, int mem);

/* GFMC_MODEL_DEX_INF only.  Undamped moments in the pair of states {|o>, |v>} of Eq. (21)-(22):
 *   |v_s> = Delta|o_s> = sum_j Delta_jo |j>,  Delta = H' - H for the trial spin proposals[s] at sites[s]  (Eq. (15))
 *   mu[s][n][alpha][beta][re,im] = <alpha| T_n(H~) |beta>,  alpha, beta in (o, v);  |v> is not normalised (mu_0(v,v) = <v|v>).
 * proposals [n_sites][3].  The paper obtains the off-diagonal elements from mixed diagonal ones (Eq. (33)-(36));
 * the doubling identity in its 2x2 form gives them directly from the same two vectors. */
int gfmc_moments_ov(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites, const double* proposals, double* mu, int mem);

/* GFMC_MODEL_DEX_INF only.  G[s][k][alpha][beta] = <alpha| 1/(H - z) |beta> in {o, v}, physical units, kernel-damped, on the
 * grid E[k] of gfmc_local_green; d(z) of Eq. (22) is [1 + G_ov][1 + G_vo] - G_oo G_vv.  E or G may be NULL. */
int gfmc_local_green_ov(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites, const double* proposals,
                        double* E, double* G, int mem);

/* GFMC_MODEL_DEX_INF only.  Forward bond amplitudes of Eq. (3) for the current configuration:
 *   Tb[d][i][re,im] = t_{i, i+e_d},  d = 0 (x), 1 (y), 2 (z);  <i|H|i+e_d> = -t * t_{i,i+e_d};  3*N complex values. */
int gfmc_hopping(gfmc_ctx* ctx, double* Tb, int mem);

/* Local 2x2 Green's function on the Chebyshev-node grid, kernel-damped (a4-a5):
 *   E[k] = a cos(pi (k+1/2)/K) + b  (physical energies, descending), k = 0..K-1
 *   G[s][k][alpha][beta][re,im] = <o_s alpha| 1/(H - z) |o_s beta>, z = E_k + i0, in physical units (= G~/a).
 * E or G may be NULL. */
int gfmc_local_green(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites, double* E, double* G, int mem);

/* Effective-action change for one trial spin per listed site, every site evaluated against the CURRENT
 * configuration (a3-a6); the configuration is not modified.  proposals [n_sites][3] are the trial spins S'
 * of sites[j]; dS [n_sites]. */
int gfmc_delta_S(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites, const double* proposals, double* dS, int mem);

/* One frozen-batch Metropolis update (a2-a7): Delta S for every listed site against the configuration at
 * call time, accept iff -Delta S > ln(uniforms[j]), then all accepted flips applied together.
 * n_sites <= max_batch_sites; sites must be distinct.  proposals [n_sites][3], uniforms [n_sites] in (0,1].
 * dS [n_sites] and accepted [n_sites] (0/1) may be NULL. */
int gfmc_update_batch(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites,
                      const double* proposals, const double* uniforms,
                      double* dS, uint8_t* accepted, int mem);

/* one chain whose frozen batches are sharded over G GPUs (start vectors are independent; PAPER.md:259-263 is the
 * paper's own, coarser level: independent chains).  Every rank holds the whole spin field (24 B x N) and its own context:
 *   gfmc_decide_batch: rows a2-a6 and the accept test of gfmc_update_batch for the rank's share of the batch, against the current
 *     configuration, which is NOT modified; same arguments and outputs as gfmc_update_batch.  GFMC_BATCH_FROZEN only
 *     (GFMC_EINVAL in GFMC_BATCH_EXACT mode: those decisions depend on each other).
 *   [one all-gather of (accepted, dS) between the ranks -- the caller's: torch.distributed / NCCL in sharded.py]
 *   gfmc_apply_flips: S_sites[j] <- proposals[j] wherever accepted[j] != 0, for the WHOLE batch (any n_sites; processed in chunks),
 *     then the bond amplitudes of GFMC_MODEL_DEX_INF are refreshed.  sites [n_sites] distinct (host lists are checked:
 *     GFMC_EINVAL on a repeat or an out-of-range site; device lists are trusted), proposals [n_sites][3], accepted [n_sites].
 * Decisions do not depend on how the batch is cut (each site is evaluated independently against the same configuration), so the
 * sharded chain has the same accept flags and the same spins, bit for bit, as the single-GPU chain; Delta S agrees to rounding
 * (the summation order of the Gram sums depends on the number of slots in a launch). */
int gfmc_decide_batch(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites,
                      const double* proposals, const double* uniforms,
                      double* dS, uint8_t* accepted, int mem);
int gfmc_apply_flips(gfmc_ctx* ctx, const int32_t* sites, int32_t n_sites,
                     const double* proposals, const uint8_t* accepted, int mem);

/* SURVEY.md 8(f) row f5, "exactness inside a batch".  The paper's Algorithm 1 is sequential: every trial is
 * evaluated with the Green's function of the current Hamiltonian.  A frozen batch (GFMC_BATCH_FROZEN) evaluates all its sites
 * against the configuration at batch start, which is off at second order in the inter-site Green's function.  In
 * GFMC_BATCH_EXACT mode gfmc_update_batch / gfmc_sweep / gfmc_run decide the sites of a batch one after the other, in list order:
 * with U the earlier ACCEPTED sites of the batch, Eq. (11) for the pair (H + Delta_U, H + Delta_U + Delta_B) gives
 *     d_B|U(z) = det_2(1_2 + G_U,BB(z) Delta_B),   G_U,BB = G_BB - G_BU Delta_U (1 + G_UU Delta_U)^-1 G_UB   (Dyson / Woodbury),
 * from the Green blocks G_XY(z) = <o_X a|1/(H - z)|o_Y b> between the sites of the batch at batch start.  Those come from cross
 * moments <o_X a|T_m(H~)|o_Y b> read out of the work vectors after every fused step; the doubling of Eq. (27)-(28) does not apply
 * to them, so a batch costs M-1 fused steps instead of M/2.  No new Chebyshev recursion is needed after an accepted flip.
 * With the exact resolvent the conditional ratios are exact; with the truncated series they agree with the sequential algorithm up
 * to truncation error: O(1/M) for the Lorentz kernel (the damped series is the resolvent at a complex energy, where the identity
 * holds), and as long as the broadening exceeds the level spacing for the Jackson kernel.
 * Requires exact_batch_sites > 0 at gfmc_create (else GFMC_ESTATE); batches larger than exact_batch_sites give GFMC_EINVAL.
 * A batch in which some Delta S is not finite, or 1 + G Delta is singular at an energy node (d_k = 0: no Woodbury update exists), is
 * abandoned with GFMC_ESTATE before any flip is written: the configuration is the one at batch start (earlier batches of the same
 * gfmc_sweep / gfmc_run call stay applied). */
int gfmc_set_batch_mode(gfmc_ctx* ctx, int mode);

/* n_sweeps Monte Carlo sweeps (Algorithm 1) with the colour-major frozen-batch schedule:
 * for each sweep, for colour c = (x+y+z) mod 2 in (0,1), the sites of colour c in increasing index order are
 * cut into consecutive batches of batch_sites (<= max_batch_sites; the last may be short); each batch is one
 * gfmc_update_batch.  batch_sites = 1 is the paper's sequential algorithm (deterministic site order).
 * Precondition of the schedule: (x+y+z) mod 2 is a proper two-colouring of the periodic lattice only for EVEN L.  At odd L the
 * wrap neighbours x = 0 and x = L-1 share a colour, so a batch may hold nearest neighbours: for GFMC_MODEL_HUND that is the same
 * kind of frozen-batch approximation as for any two sites (second order in the inter-site Green's function, larger for
 * neighbours); for GFMC_MODEL_DEX_INF two neighbouring flips change the SAME bond t_ij, the joint Delta is not the sum of the
 * single-site Deltas, and gfmc_sweep / gfmc_run return GFMC_EINVAL for odd L with batch_sites > 1.
 * proposals [n_sweeps][N][3] and uniforms [n_sweeps][N] are indexed by SITE; randomness never lives in the library.
 * Outputs (each may be NULL): dS_log, accept_log [n_sweeps][N] indexed by site; magnetization [n_sweeps]
 * = |sum_i S_i|/N after each sweep (Alg. 1 line 15); n_accepted [n_sweeps]. */
int gfmc_sweep(gfmc_ctx* ctx, int32_t n_sweeps, int32_t batch_sites,
               const double* proposals, const double* uniforms,
               double* dS_log, uint8_t* accept_log,
               double* magnetization, int64_t* n_accepted, int mem);

/* Algorithm 1 with the trial moves drawn by the library.
 * The paper says "change the spin randomly" (line 4) and compares with rand() (line 10) without naming
 * a generator; reading f3-1 fixes the counter-based Philox4x32-10 with key = (seed mod 2^32, seed div 2^32) and
 * counter = (site, sweep mod 2^32, stream, sweep div 2^32): stream 0 gives (u1, u2), stream 1 gives u3, each
 * floor((w_even 2^32 + w_odd) / 2^11) 2^-53 in [0,1); trial spin S' = (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z) with
 * z = 2 u1 - 1, phi = 2 pi u2 (uniform on the sphere, independent of the current spin); acceptance uniform 1 - u3 in (0,1].
 * The numbers depend on (seed, sweep, site) only, so (spins, seed, next sweep index) is a complete checkpoint of a chain.
 *
 * gfmc_random_proposals: writes proposals [N][3] and uniforms [N] of sweep `sweep` (indexed by site) -- exactly the arrays that
 *   gfmc_run feeds to the sweep; exposed so that they can be checked and so that gfmc_sweep can replay a gfmc_run chain.
 * gfmc_run: sweeps first_sweep .. first_sweep + n_sweeps - 1 with the schedule of gfmc_sweep; trial moves are generated on the
 *   device, only magnetization [n_sweeps] and n_accepted [n_sweeps] (either may be NULL) are written (mem: where they live).
 * Errors: GFMC_EINVAL (NULL / negative sweep index / batch_sites out of range), GFMC_ESTATE (spins not set), GFMC_ECUDA. */
int gfmc_random_proposals(gfmc_ctx* ctx, uint64_t seed, int64_t sweep, double* proposals, double* uniforms, int mem);
/* Changes the temperature T (> 0, finite; else GFMC_EINVAL) used by every later Delta S_eff (beta = 1/T in Eq. (14));
 * moments and Green's functions do not depend on it.  Lets one context anneal through the temperatures of an M(T) curve
 * (Fig. 4 at 378). */
int gfmc_set_temperature(gfmc_ctx* ctx, double T);
int gfmc_run(gfmc_ctx* ctx, uint64_t seed, int64_t first_sweep, int32_t n_sweeps, int32_t batch_sites,
             double* magnetization, int64_t* n_accepted, int mem);
/* Alg. 1 lines 16-17 ("M <- M + m" ... "return M/S") for the sweeps of the most recent successful gfmc_run on
 * this context, accumulated on the device sweep by sweep: mean of m = |sum_i S_i|/N over the S sweeps, its naive standard error
 * sqrt(sum (m - mean)^2 / (S-1) / S) (NaN for S = 1; the sweeps of a chain are correlated, so this is a lower bound), and the
 * acceptance ratio (accepted flips / (S N)).  HOST output pointers, each may be NULL.  GFMC_ESTATE if there is no such run. */
int gfmc_run_summary(gfmc_ctx* ctx, double* mean_magnetization, double* stderr_magnetization, double* acceptance, int64_t* n_sweeps);

/* |sum_i S_i| / N of the current configuration (a8). */
int gfmc_magnetization(gfmc_ctx* ctx, double* m);

/* Moments without a context and WITHOUT ANY ALLOCATION -- for callers that may not allocate device memory when they need the
 * result: a process whose own pool allocator took the whole GPU at start-up (cudaMalloc then fails or disturbs the pool), a
 * thread running beside another thread's global-mode stream capture (an allocation call would break that capture), a loop
 * that cannot afford the device-wide synchronisation hidden in cudaMalloc / cudaFree.  gfmc_create allocates or needs a sized
 * workspace; this call needs neither.  It calls no cudaMalloc, cudaFree or other allocating routine.
 *
 * Computes exactly what gfmc_moments computes for GFMC_MODEL_HUND, ph_symmetry = 0 (same kernels, same rounding):
 *   mu[s][n][alpha][beta][re,im] = <o_s alpha| T_n(H~) |o_s beta>,  n = 0..M-1,  a = 6|t| + sqrt(2)|J_H|   Eq. (25)-(28)
 * with the vectors resident in shared memory, so 2 <= L <= 12 (GFMC_STATIC_MAX_L).  The scratch memory of that path (an SoA copy
 * of the spins, and the Gram sums between the recursion kernel and the moment read-out) is a fixed array inside the library image:
 * 8 * (6144 + 8 * GFMC_STATIC_MAX_STEP_SITES) bytes = 4.05 MiB on every device that loads libgfmc.so, held until the process exits.
 * Limit: (M/2) * n_sites <= GFMC_STATIC_MAX_STEP_SITES (e.g. M = 256 with 512 sites, M = 64 with 2048); beyond it, or for L > 12,
 * the call returns GFMC_EINVAL and changes nothing -- split the site list, or use gfmc_create + gfmc_moments.
 *
 * Arguments: device = CUDA ordinal (made current for the call, the previous one restored); stream = cudaStream_t to launch on (NULL =
 * legacy default stream); S [L^3][3] spins, sites [n_sites] in 0..L^3-1 (any order, repeats allowed), mu [n_sites][M][2][2] complex:
 * all three are DEVICE pointers on `device`, caller-owned, trusted (not validated), read / written only during the call.
 * Synchronous: the stream has drained on return.  n_sites = 0 is allowed and does nothing.
 * First call on a device: looks up the device address of the scratch array and opts the kernels in to large shared memory (this
 * also makes the CUDA runtime load the library's device code).  Make that first call before any stream capture is begun.
 * Sharing: all calls on a device use the same scratch array, which keeps whatever the last call left there.  Nothing in it needs
 * to start at zero (every entry a call reads, that call wrote first).  Calls that overlap on the GPU -- two threads, two streams --
 * race on it; serialise them.  Contexts made by gfmc_create never touch the array.
 * Errors: GFMC_EINVAL (sizes beyond the maximum, L / M / device out of range, NULL), GFMC_ECUDA (no sm_100 device, a CUDA call
 * failed); text from gfmc_moments_static_error() (per thread, valid until that thread's next call). */
#define GFMC_STATIC_MAX_L           12
#define GFMC_STATIC_MAX_STEP_SITES  65536
int gfmc_moments_static(int32_t device, void* stream, int32_t L, int32_t M, double t, double JH,
                        const double* S, const int32_t* sites, int32_t n_sites, double* mu);
const char* gfmc_moments_static_error(void);

/* Instrumentation for benchmarks (not part of the method): counts of kernels launched by this context since
 * creation (index 0: fused Chebyshev step kernels, 1: all other kernels), and device time in milliseconds
 * spent in the Chebyshev step loops of the most recent call, measured with CUDA events on the context's stream, together with
 * the number of fused steps those loops ran.  At most the first 64 batches of a call are timed (the rest of a long sweep is
 * not, and is not counted in n_steps either), so ms / n_steps is always the average duration of a fused step.  With
 * GFMC_FLAG_TWO_STEP a launch performs two steps: n_steps still counts STEPS, gfmc_launch_counts counts launches (M/4 per batch). */
int gfmc_launch_counts(const gfmc_ctx* ctx, int64_t counts[2]);
int gfmc_last_step_loop_ms(const gfmc_ctx* ctx, double* ms, int64_t* n_steps);
/* Start vectors propagated by the most recent batch of the most recent call and the algorithmic bytes of one fused step over
 * them (48 B per complex element: read r_{m-1}, read r_{m-2}, write r_m). */
int gfmc_last_step_loop_vectors(const gfmc_ctx* ctx, int64_t* n_vectors, int64_t* bytes_per_step);

const char* gfmc_last_error(const gfmc_ctx* ctx);
const char* gfmc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GFMC_H */
