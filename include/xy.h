/* xy.h -- C ABI of the B200-native Monte Carlo step of the 3-D classical XY model
 *
 *     H = - sum_<ij> cos(theta_i - theta_j)        L x L x L periodic cubic lattice, J = k_B = 1
 *
 * over R parallel-tempering replicas, after arXiv:1211.0780 (cited as P:<line of PAPER.md>).
 * One Monte Carlo step is
 *
 *     xy_metropolis_sweep -> xy_overrelax_sweep -> xy_measure -> xy_pt_exchange
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  The
 * readings of the paper that these calls implement (proposal rule, colour order, RNG keying,
 * pair selection, ...) are listed in DESIGN.md section 2 (R1..R17).
 *
 * Vocabulary.  N = L^3 sites.  A *slot* r is a physical spin array (it never moves); a *rank*
 * k is an index into the caller's betas[] (a temperature).  Replica exchange permutes which
 * slot carries which rank (slot_at_rank), never the spins (R11).  Natural layout means
 * float theta[R][L][L][L] indexed [slot][z][y][x], x fastest, angles in radians in [0, 2 pi].
 * Inside the library the state is colour-split: colour = (x+y+z)&1, 0 = black (updated
 * first, R3); theta_c[slot][z][y][x>>1], two arrays of R*N/2 floats.
 *
 * Conventions.  Functions returning int return XY_OK (0) or a negative XY_ERR_*; they never
 * throw, abort or print.  xy_last_error() gives a thread-local message for the last failing
 * call.  Pointers are HOST pointers unless the parameter says "device".  A context is not
 * thread-safe.  All device work is enqueued on the attached stream, in call order; only calls
 * that return host data synchronise it.  L must be a multiple of 8 (128-bit rows), R >= 1.
 */
#ifndef XY_H_
#define XY_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct xy_ctx xy_ctx;

enum {
    XY_OK = 0,
    XY_ERR_INVALID_ARG = -1,  /* bad L/R/pointer/beta/option; nothing was enqueued             */
    XY_ERR_CUDA = -2,         /* a CUDA call failed (message in xy_last_error)                 */
    XY_ERR_NOT_ATTACHED = -3, /* the context has no device buffers yet (call xy_attach)        */
    XY_ERR_NO_DEVICE = -4     /* no usable sm_100 device: the library never falls back to CPU  */
};

#define XY_NUM_OBS 5 /* E, Mx, My, |M|^2, |M|^4 */

/* Tunables for xy_set_option (all optional; defaults are chosen from L and R). */
enum {
    XY_OPT_TILE_Y = 1,     /* rows of one colour per thread block (must divide L, TILE_Y*L/8 <= 352) */
    XY_OPT_TILE_Z = 2,     /* planes a thread block marches through (must divide L)                  */
    XY_OPT_TRACE = 3,      /* 1: xy_metropolis_sweep also records its fast-path acceptance probability
                              per site (test hook; allocates R*N floats inside the library)         */
    XY_OPT_FUSED_MEASURE = 4, /* 1 (default): the white over-relaxation pass also accumulates the
                              observables of the state it leaves behind, so xy_measure / xy_pt_exchange
                              after xy_overrelax_sweep read no spins; 0: always the standalone reduction */
    XY_OPT_PROFILE = 5,    /* 1: bracket every kernel launch with a CUDA-event pair on the attached
                              stream; xy_get_kernel_times returns the per-class device times         */
    XY_OPT_GENERIC_KERNEL = 6, /* 1: always run the colour-pass kernel that reads the row geometry at run
                              time, also for L = 32, 64, 128, 160 where a compile-time variant exists  */
    XY_OPT_OR_PER_MCS = 7, /* over-relaxation sweeps per Monte Carlo step of xy_mcs (default 1, P:30;
                              P:43 "after several sweeps": microcanonical sweeps are cheap decorrelation) */
    XY_OPT_CUDA_GRAPH = 8, /* 1 (default): xy_mcs replays one captured CUDA graph per step from its second
                              step on (counters live on the device); 0: every kernel is launched eagerly  */
    XY_OPT_RESIDENT = 9,   /* 1 (default): for small lattices (L = 8 ... 48, R <= 512, everything co-resident) xy_mcs
                              runs all its steps in ONE persistent launch with the spins resident in shared
                              memory.  Same site arithmetic and Philox keying as the per-pass kernels:
                              the spins after a call are bitwise theirs, the observables agree within the reduction's
                              rounding (their fp32 terms are grouped differently).  The exchange compares log(u) < x
                              where the per-pass kernels compare u < exp(x), on energies that differ by that rounding:
                              a decision within about 1e-8 of its threshold can fall the other way (inside the 1e-6
                              window of P4), and from such a step on the two trajectories part -- both are valid, only
                              bitwise equality between the two paths is lost (never seen in the tests' runs).
                              While this path is taken, XY_OPT_TILE_Y / TILE_Z / GENERIC_KERNEL / FUSED_MEASURE /
                              CUDA_GRAPH / SLOT_CHUNK do not apply to xy_mcs (they still govern the sweep-by-sweep
                              calls); XY_OPT_TRACE = 1 forces the per-pass kernels (xy_get_resident_plan says which
                              path xy_mcs takes).  0: always the per-pass kernels                                */
    XY_OPT_SLOT_CHUNK = 10 /* K > 0: xy_mcs runs the four colour passes of K slots at a time back to back (launches
                              over slots [0,K), [K,2K), ...) so that a chunk's spins stay in the 126 MB L2 between
                              its passes: 8 instead of 24 B of HBM traffic per site and step (SURVEY 8(f) f2 for
                              lattices too large for shared memory).  Same kernels, bitwise the same results.
                              0 (default): every pass runs over all slots at once (faster: DESIGN.md section 6) */
};

/* Kernel classes reported by xy_get_kernel_times. */
#define XY_NUM_KERNEL_CLASSES 8
enum {
    XY_K_METROPOLIS = 0, /* one Metropolis colour pass over all slots (a2)                         */
    XY_K_OVERRELAX = 1,  /* one over-relaxation colour pass over all slots (a3)                    */
    XY_K_MEASURE = 2,    /* the observable reduction over all slots (a4, first stage)              */
    XY_K_FINALIZE = 3,   /* a4 final stage: per-slot sums in fixed order, by-rank output           */
    XY_K_PT = 4,         /* the replica-exchange kernel (a5)                                       */
    XY_K_OTHER = 5,      /* init, fill, layout conversion                                          */
    XY_K_FIXUP = 6,      /* a2: fp64 settlement of the close Metropolis decisions of one colour pass */
    XY_K_RESIDENT = 7    /* a2..a5 of n whole steps in one persistent launch (small lattices, XY_OPT_RESIDENT) */
};

/* ---- lifetime ------------------------------------------------------------------------------ */

/* Creates the host-side description of one (L, R) system: copies betas[0..R-1] (rank order; need
 * not be sorted -- adjacency for replica exchange is adjacency in this array), stores the
 * Philox key `seed`, sets slot_at_rank[k] = k and all counters to 0.  Allocates nothing on the
 * device.  Returns NULL on invalid arguments (L < 8 or L % 8 != 0, R < 1, NULL or non-finite
 * betas); the reason is in xy_last_error().  [north_star: xy_create(L, R, betas, seed)] */
xy_ctx* xy_create(int L, int R, const double* betas, uint64_t seed);

/* Frees the context and whatever it allocated itself (on the context's device, whichever device is current);
 * attached caller-owned buffers and the stream are not touched.  NULL is allowed. */
void xy_destroy(xy_ctx* ctx);

/* Bytes of device memory a context of this shape needs: the colour-split state (R*N floats)
 * and the workspace (reduction partials, results, permutation, beta labels, acceptance
 * counters, one natural-layout staging slot).  0 on invalid (L, R). */
size_t xy_state_bytes(int L, int R);
size_t xy_workspace_bytes(int L, int R);

/* Binds device memory and a stream.  d_state / d_workspace: DEVICE pointers, 256-byte aligned,
 * of at least xy_state_bytes / xy_workspace_bytes, on the CURRENT device, owned by the caller
 * (PyTorch) and required to outlive the context.  A caller's stream must belong to the current device too
 * (XY_ERR_INVALID_ARG otherwise).  The context is bound to the device that is
 * current at this call: every later entry point switches to it for its own duration and restores
 * the caller's current device.  Either buffer may be NULL, in which case the library cudaMallocs and owns it.
 * cuda_stream: a cudaStream_t; NULL = the library creates a blocking stream of its own, which is
 * implicitly ordered with the legacy default stream (that one cannot be captured into a CUDA graph).  Uploads the beta labels and
 * the identity permutation; the spin state is undefined until xy_init_* or xy_set_state. */
int xy_attach(xy_ctx* ctx, void* d_state, void* d_workspace, void* cuda_stream);

/* ---- state (a0) ---------------------------------------------------------------------------- */

/* Random start: theta[r][i] = fl32(2pi_f * u24(W[i&3])), W = Philox4x32-10(key = seed,
 * counter = (i>>2, r, 0, stream 0)), i = x + L*(y + L*z)  [configs: "random-start angles from
 * seed"; R12, R17].  Ordered start: every angle = theta0 [config 4].  Both reset the cached
 * observables; neither touches counters or the permutation. */
int xy_init_random(xy_ctx* ctx);
int xy_init_ordered(xy_ctx* ctx, float theta0);

/* Copies a natural-layout configuration in / out (R*N floats).  on_device = 0: `natural` is a
 * host pointer (pinned memory makes the copy asynchronous-capable; the call synchronises
 * before returning for xy_get_state, and before the host buffer may be reused for
 * xy_set_state); on_device = 1: a device pointer readable from the attached stream, no
 * synchronisation.  The layout conversion runs in a kernel.  The kernels' stated errors hold for
 * angles in [0, 2 pi]: xy_set_state reduces any finite angle outside that range modulo 2 pi
 * (angles inside it are stored bit for bit); a NaN or infinite angle is stored as 0. */
int xy_set_state(xy_ctx* ctx, const float* natural, int on_device);
int xy_get_state(xy_ctx* ctx, float* natural, int on_device);

/* ---- the Monte Carlo step (a2..a5) ----------------------------------------------------------- */

/* One checkerboard Metropolis sweep over all R slots: every black site, then every white site
 * [P:30, Fig. 2 P:36].  For site i of slot r with local field h = sum over the six neighbours
 * of (cos, sin) [P:23-28 Eq. 1]:  W = Philox(counter = (i>>2, r, n_met, 1 + colour)),
 * p = (i>>1)&1, theta' = fl32(2pi_f * u24(W[2p])), dE = -h.(S(theta') - S(theta)),
 * accept iff u24(W[2p+1]) < exp(-fl32(beta_of_slot[r]) * dE)  [R1, R2, R12, R13].
 * The decision is taken in fp32 fast arithmetic when it is clear.  When |u - p_fast| is inside the
 * window |beta| * 4e-5 + 1.5e-6 (the derived bound of the fast path's error, csrc/xy_device.cuh) the
 * site is appended to a device queue and settled by met_fixup_kernel in fp64 from the stored
 * angles right after the colour pass (for very large |beta|, where most decisions are close, in
 * the pass itself), so every decision equals the fp64 definition.  Accepted
 * angles are bit-identical to the definition.  Should a pass ever produce more close decisions
 * than the queue holds, a sticky flag makes every later synchronising call return XY_ERR_CUDA
 * ("queue overflowed") until the context is attached again: results are then not exact.  ++n_met. */
int xy_metropolis_sweep(xy_ctx* ctx);

/* One checkerboard over-relaxation sweep, black then white: theta' = 2*atan2(h_y, h_x) - theta
 * reduced to [0, 2pi); unchanged if h = 0  [P:38-43 Eq. 2; R4-R7].  fp32 arithmetic with a
 * stated field error.  With XY_OPT_FUSED_MEASURE (default) the white pass
 * also produces the observables of the new state.  ++n_or. */
int xy_overrelax_sweep(xy_ctx* ctx);

/* Observables of the current state, out[R][5] = E, Mx, My, |M|^2, |M|^4 indexed by RANK k
 * [P:52-56 Eqs. 4-5; E_n of Eq. 3; R14, R15]: E = -sum_bonds cos(theta_i - theta_j)
 * (3N bonds), Mx = sum cos, My = sum sin; fp32 site terms, fp64 fixed-order accumulation
 * (deterministic run to run).  out: host pointer, R*5 doubles, written after a stream
 * synchronise; NULL = only enqueue the reduction (results stay on the device for
 * xy_pt_exchange).  Re-uses cached results when the state has not changed since they were
 * produced. */
int xy_measure(xy_ctx* ctx, double* out);

/* The six sums behind the spin-stiffness estimator [P:58-60 Eq. 6] of the current state,
 * out[R][6] = Cx, Cy, Cz, Sx, Sy, Sz indexed by RANK k, with, over the N bonds (i, i+mu) of
 * direction mu,  C_mu = sum cos(theta_i - theta_{i+mu}),  S_mu = sum sin(theta_i - theta_{i+mu}).
 * Eq. 6 is rho_s = 1/(3N) sum_mu [ <C_mu> - beta <S_mu^2> ], host arithmetic on the time series;
 * E = -(Cx + Cy + Cz).  fp32 bond terms, fp64 fixed-order accumulation; one pass over the spins
 * (4 B per site).  out: host pointer, R*6 doubles, written after a stream synchronise. */
int xy_measure_stiffness(xy_ctx* ctx, double* out);

/* One replica exchange [P:45-50 Eq. 3; R8-R11]: for k = n_pt mod 2, k+2, ... with k+1 < R,
 * a = slot_at_rank[k], b = slot_at_rank[k+1], u = W[0] * 2^-32 with
 * W = Philox(counter = (k, 0, n_pt, 3)); accept iff u < exp((betas[k]-betas[k+1])*(E_a-E_b)),
 * in fp64; on accept the two slots exchange their rank / beta label.  Uses the cached
 * energies, running the reduction first if they are stale.  ++n_pt. */
int xy_pt_exchange(xy_ctx* ctx);

/* n_mcs repetitions of (Metropolis sweep, XY_OPT_OR_PER_MCS over-relaxation sweeps, measure, PT exchange) [P:30],
 * enqueued without host synchronisation.  series: DEVICE pointer to n_mcs*R*5 doubles that
 * receives the by-rank observables of every step (measured before that step's exchange, R14),
 * or NULL. */
int xy_mcs(xy_ctx* ctx, int n_mcs, double* d_series);

/* ---- bookkeeping ----------------------------------------------------------------------------- */

int xy_get_perm(xy_ctx* ctx, int* slot_at_rank /* R, out */);         /* synchronises */
int xy_set_perm(xy_ctx* ctx, const int* slot_at_rank /* R, a permutation */);
int xy_get_beta_of_slot(xy_ctx* ctx, double* beta_of_slot /* R, out */); /* synchronises */
/* Replaces the temperature ladder (R values, rank order): rank k keeps the slot it holds and gets betas[k].  For
 * tuning a ladder towards temperature-independent swap acceptance [P:62] from xy_get_accept_counts.  Synchronises. */
int xy_set_betas(xy_ctx* ctx, const double* betas);
int xy_get_counters(xy_ctx* ctx, uint32_t counters[3] /* n_met, n_or, n_pt */);
int xy_set_counters(xy_ctx* ctx, const uint32_t counters[3]);
/* Accepted Metropolis proposals per SLOT and accepted swaps per pair (k, k+1) since attach;
 * either pointer may be NULL.  Synchronises. */
int xy_get_accept_counts(xy_ctx* ctx, uint64_t* met_acc /* R */, uint64_t* pt_acc /* R-1 */);
/* Number of Metropolis decisions that took the fp64 re-evaluation since attach.  Synchronises. */
int xy_get_exact_path_count(xy_ctx* ctx, uint64_t* n);
int xy_set_option(xy_ctx* ctx, int option, int value);
int xy_get_option(xy_ctx* ctx, int option, int* value);
/* How xy_mcs will run on this context (XY_OPT_RESIDENT): out[0] = 1 if all steps of a call run in one persistent
 * launch with the spins resident in shared memory, else 0 (per-pass kernels: no plan fits, XY_OPT_RESIDENT = 0 or XY_OPT_TRACE = 1); out[1] = slots per thread block,
 * out[2] = thread blocks (cluster size) per slot, out[3] = threads per block, out[4] = blocks, out[5] = dynamic
 * shared memory per block in bytes.  The plan needs the device: call after xy_attach. */
int xy_get_resident_plan(xy_ctx* ctx, int out[6]);
/* Number of kernels this context has launched since attach (bench.py's gpu_launches). */
int xy_get_launch_count(xy_ctx* ctx, uint64_t* n);
/* With XY_OPT_PROFILE = 1: device time in milliseconds (CUDA events on the attached stream) and
 * number of launches per kernel class since the previous call; ms and launches have
 * XY_NUM_KERNEL_CLASSES entries.  Synchronises, then resets the accumulators. */
int xy_get_kernel_times(xy_ctx* ctx, double* ms, uint64_t* launches);
int xy_synchronize(xy_ctx* ctx);
const char* xy_last_error(void);

/* ---- the observable reduction for callers that cannot allocate device memory ----------------- */

/* Capacity of the library's built-in scratch area used by xy_measure_static, in bytes. */
#define XY_STATIC_SCRATCH_BYTES (1u << 20)

/* E, Mx, My, |M|^2, |M|^4 [P:52-56 Eqs. 4-5] of R spin configurations, WITHOUT a context, a workspace or any
 * allocation: the call neither runs cudaMalloc / cudaFree nor any library routine that allocates.
 *
 * Who needs this.  Every other entry point works on an xy_ctx whose workspace (xy_workspace_bytes: 50 MB at
 * L = 160 x 64) somebody has to allocate -- the caller before xy_attach, or xy_attach itself with cudaMalloc.
 * Some code that holds a spin state can do neither: an analysis or monitoring hook that is only lent the state
 * buffer by a simulation which has already given the rest of the GPU to its own memory pool (a raw cudaMalloc
 * then fails, or is forbidden by the host program's rules); a service loop that must not stall, where
 * cudaMalloc / cudaFree are unacceptable because they synchronise the whole device; a process whose memory
 * budget is fixed at start-up.  For them the reduction's scratch (the per-tile partial sums between its two
 * kernels) lives in an array compiled into the library, XY_STATIC_SCRATCH_BYTES = 1 MiB of device memory that
 * every GPU holds from the moment it loads this library's code until the process exits.
 *
 * d_state:  DEVICE pointer, the colour-split state exactly as the library keeps it in the d_state buffer of
 *           xy_attach (top of this file: black half-lattices of all R slots, then the white ones; R*N floats,
 *           angles in [0, 2 pi]), 16-byte aligned, on the CURRENT device.  Read only.
 * d_out:    DEVICE pointer, R*5 doubles, written as out[slot][5] -- indexed by SLOT, not by rank: there is no
 *           context here and therefore no permutation (xy_get_perm maps ranks to slots).
 * cuda_stream: a cudaStream_t on the current device (NULL = the default stream).  The two kernels are
 *           enqueued there; the call does not synchronise and d_out is valid once the stream has reached
 *           the end of this call's work.
 *
 * Same kernels and arithmetic as xy_measure (fp32 site terms, fp64 fixed-order sums, deterministic); the
 * tiles are the library's defaults for (L, R) and always the run-time-geometry kernel, so against xy_measure
 * on a context with other tiles the sums differ by rounding only (well inside 1e-6 * 3N).
 *
 * Limit.  The scratch need is 24 bytes x R x (thread-block tiles per replica).  All five BASELINE configs and
 * the paper's families need under 64 KiB; a shape that needs more than XY_STATIC_SCRATCH_BYTES (e.g. L = 8
 * with R > 43690) is refused with XY_ERR_INVALID_ARG and a message that names need and capacity; nothing is
 * enqueued.  Use xy_measure on a context for those.
 *
 * First call on a device.  The first call made while a given device is current looks up the device address
 * of the built-in array and raises the kernel's shared-memory limit, once per device.  That set-up is not
 * stream work: make this first call at start-up, before any stream capture is begun on that device.
 *
 * Sharing.  There is ONE scratch array per device and every call uses it, whatever the stream or host
 * thread.  It keeps whatever the previous call left there; that is harmless because each call's first kernel
 * overwrites every entry its second kernel reads (nothing has to start at zero, nothing is cleared).  But two
 * calls whose kernels can overlap on the GPU -- different streams without an event between them, or two host
 * threads -- race on it and both get garbage: keep calls on one stream, or order them with events.
 *
 * Errors: XY_ERR_INVALID_ARG (shape, size beyond the scratch, NULL / misaligned / non-device / wrong-device
 * pointer), XY_ERR_NO_DEVICE (no sm_100 device current), XY_ERR_CUDA. */
int xy_measure_static(const float* d_state, int L, int R, double* d_out, void* cuda_stream);

/* ---- test hooks (stated-error measurements; not part of the Monte Carlo step) ---------------- */

/* With XY_OPT_TRACE = 1: the fast-path acceptance probability min(p_fast, FLT_MAX) of every site
 * in the last xy_metropolis_sweep, natural layout, host pointer, R*N floats.  Synchronises. */
int xy_debug_get_trace(xy_ctx* ctx, float* natural);
/* Evaluate the kernels' device math on n DEVICE floats (stream = cudaStream_t or NULL):
 * fast sin/cos of x[i]; fast atan2(y[i], x[i]) in [0, 2pi); Philox words of n counters. */
int xy_debug_sincos(const float* d_x, float* d_cos, float* d_sin, size_t n, void* cuda_stream);
/* the fp64 sin / cos of the settlement of close Metropolis decisions, for n DEVICE doubles in [0, 2 pi] */
int xy_debug_sincos64(const double* d_x, double* d_cos, double* d_sin, size_t n, void* cuda_stream);
int xy_debug_atan2(const float* d_y, const float* d_x, float* d_phi, size_t n, void* cuda_stream);
int xy_debug_philox(const uint32_t* d_ctr /* n*4 */, uint32_t key0, uint32_t key1,
                    uint32_t* d_out /* n*4 */, size_t n, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* XY_H_ */
