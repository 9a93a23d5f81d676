/* chisao.h -- C ABI of libchisao: one CHISAO convergence/anti-convergence oscillation cycle over a whole
 * population, as hand-written sm_100a CUDA kernels (fp32 on device).
 *
 * Method: arxiv/paper_2606_26164 (/root/reference/PAPER.md at build time; cited below as PAPER.md:<line>).
 *   Problem statement  PAPER.md:62-69  (population {x_i} in a bounded box Theta, value-only f, returns modes)
 *   Algorithm 1        PAPER.md:141-176 (for k = 1..n_osc: phases 1-3 always, 4-6 iff k < n_osc)
 *   Phases 1-6         PAPER.md:75-131  (Eq. 2-6), defaults in Table 1
 * Readings of silent/garbled passages are listed in DESIGN.md ("Readings", R-1..R-17).
 *
 * Conventions
 *   - Every entry point returns 0 on success or a negative CHISAO_E_* code; no exception crosses the ABI;
 *     chisao_last_error() returns a static/ctx-owned string describing the last failure.
 *   - Pointers named *_dev are DEVICE pointers owned by the caller for the life of the context (the
 *     library never allocates or frees device memory).  Pointers inside chisao_objective / chisao_config
 *     are HOST pointers, copied during chisao_init (may be freed afterwards).
 *   - `stream` is a cudaStream_t passed as void*; every kernel and copy is enqueued on it.
 *   - A context is not thread-safe.  There is no CPU fallback: without a CUDA device every call that
 *     touches the device returns CHISAO_E_CUDA.
 */
#ifndef CHISAO_H
#define CHISAO_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CHISAO_OK            0
#define CHISAO_E_INVALID    -1   /* bad argument / unsupported configuration */
#define CHISAO_E_WORKSPACE  -2   /* workspace too small or misaligned */
#define CHISAO_E_CAPACITY   -3   /* output capacity too small (chisao_modes) */
#define CHISAO_E_CUDA       -4   /* CUDA runtime error (see chisao_last_error) */
#define CHISAO_E_STATE      -5   /* call not valid in the current state (e.g. step past n_osc) */

#if defined(__GNUC__)
#define CHISAO_API __attribute__((visibility("default")))
#else
#define CHISAO_API
#endif

#define CHISAO_MAX_D        64   /* d <= 64 */
#define CHISAO_MAX_M        16   /* L-BFGS memory m <= 16 (paper: m = 10) */

typedef struct chisao_ctx chisao_ctx;   /* opaque; host-allocated by chisao_init, freed by chisao_destroy */

/* Objective families (value-only black boxes; BASELINE.json configs C1..C5). */
typedef enum {
  CHISAO_OBJ_GMM_ISO  = 0,  /* log sum_k w_k N(x; mu_k, sigma^2 I)             (App. D) */
  CHISAO_OBJ_GMM_DIAG = 1,  /* log sum_k w_k N(x; mu_k, diag(sigma_k^2))                              */
  CHISAO_OBJ_GMM_FULL = 2,  /* log sum_k w_k N(x; mu_k, Sigma_k), Sigma_k^-1 = W_k^T W_k              */
  CHISAO_OBJ_RFF      = 3,  /* -s0 ||x||^2 + sum_j a_j cos(w_j . x + b_j)                             */
  CHISAO_OBJ_QUAD     = 4,  /* -1/2 ||W (x - c)||^2                                                   */
  /* parameter-free benchmark functions of the paper's Appendix D, negated for maximisation;
     K must be 1, the parameter pointers are ignored (may be null) */
  CHISAO_OBJ_RASTRIGIN       = 5,   /* -[10 d + sum (x^2 - 10 cos(2 pi x))] */
  CHISAO_OBJ_ACKLEY          = 6,   /* a = 20, b = 0.2, c = 2 pi */
  CHISAO_OBJ_SCHWEFEL        = 7,   /* -[418.9829 d - sum x sin(sqrt|x|)] */
  CHISAO_OBJ_STYBLINSKI_TANG = 8,   /* -1/2 sum (x^4 - 16 x^2 + 5 x) */
  CHISAO_OBJ_MICHALEWICZ     = 9,   /* sum sin(x_i) sin^20(i x_i^2 / pi) */
  CHISAO_OBJ_TRID            = 10,  /* -[sum (x_i - 1)^2 - sum x_i x_{i-1}] */
  CHISAO_OBJ_BUKIN6          = 11   /* -[100 sqrt|y - 0.01 x^2| + 0.01 |x + 10|], d = 2 */
} chisao_objective_id;

typedef struct {            /* all arrays HOST, fp32, row-major; copied at init */
  int32_t id, d, K;         /* K = #components (GMM) / #features (RFF) / 1 (QUAD) */
  const float *means;       /* GMM*: [K][d] mu_k;  QUAD: [d] c;  RFF: unused (may be NULL) */
  const float *mats;        /* ISO: [1] sigma;  DIAG: [K][d] 1/sigma_kj;  FULL: [K][d][d] W_k (row r, col c);
                               RFF: [K][d] w_j;  QUAD: [d][d] W */
  const float *vec_a;       /* GMM*: [K] log w_k + log normaliser;  RFF: [K] a_j;  QUAD: unused */
  const float *vec_b;       /* RFF: [K] b_j; else NULL */
  float scalar0;            /* RFF: s0 (1/50) */
  float sigma_noise;        /* additive evaluation noise f~ = f + N(0, sigma_noise^2); 0 = none */
} chisao_objective;

typedef struct {
  int32_t d, N;             /* dimension (1..64) and population size (>= 0) */
  const float *lo, *hi;     /* HOST [d] box bounds of Theta ("bounded domain") */
  int32_t n_osc, n_conv, n_anti, n_cloud;        /* Alg. 1 `Require`, Table 1 */
  int32_t hlc_M;            /* Hands-Like-Clouds draws per step (paper K, north_star M) */
  int32_t lbfgs_m;          /* L-BFGS memory, 1..CHISAO_MAX_M */
  int32_t ls_max;           /* backtracking trials after the first (R-4), 0..30 */
  int32_t reseed_cands;     /* Repulse-Monkey candidates per slot (R-8), 1..16 */
  float fd_h;               /* central finite-difference step (R-1) */
  float eps_grad, eps_dup, log_delta;            /* Eq. 3 / Eq. 4 thresholds */
  float mu, alpha_anti;     /* Eq. 6 momentum and step */
  float eta_hlc, sigma_s;   /* HLC step size and smoothing scale; sigma_s < 0: auto-estimate
                               sigma = |sigma_s| * std of the unfrozen samples (paper default c = 0.1; R-18) */
  float ls_c1, ls_shrink;   /* Armijo constant and backtracking factor (R-4) */
  int32_t hlc_baseline;     /* 0: literal estimator; 1: subtract the mean of the M values (R-11);
                               2: the paper's Eq. 5 form, mean of M FD gradients at perturbed points */
  uint32_t phase_mask;      /* bit p (p = 3..6) enables phase p; 0xFFFFFFFF = full algorithm */
  uint64_t seed;            /* Philox key (R-15) */
} chisao_config;

typedef struct {
  int32_t cycle, n_stuck, k_lost, n_active;
  int32_t reseed_strategy;  /* 0 none, 1 Repulse Monkey, 2 Golden Rooster, 3 uniform refill */
  int32_t gr_enabled;
  uint64_t evals[8];        /* objective evaluations: [0] cycle-start centre+FD, [1] line search,
                               [2] L-BFGS FD gradients, [5] HLC, [6] anti-convergence (cumulative);
                               [7] is not a count of evaluations: algorithmic HBM bytes moved by the L-BFGS
                               two-loop kernel (history pairs, g, x read; p, x_t written), for the roofline */
  float f_max;
} chisao_stats;

/* State fields for chisao_get_state / chisao_set_state.  Exchanged through HOST buffers, fp32 unless noted. */
enum {
  CHISAO_X = 0,        /* [N][d] */
  CHISAO_F = 1,        /* [N] */
  CHISAO_G = 2,        /* [N][d] */
  CHISAO_V = 3,        /* [N][d] */
  CHISAO_STUCK = 4,    /* [N] u8 */
  CHISAO_REMOVED = 5,  /* [N] u8 */
  CHISAO_HIST_S = 6,   /* [m][N][d], slot 0 = oldest stored pair */
  CHISAO_HIST_Y = 7,   /* [m][N][d] */
  CHISAO_HIST_LEN = 8, /* [N] i32 */
  CHISAO_STALLED = 9,  /* [N] u8 */
  CHISAO_CTRL = 10,    /* i32[8]: cycle, gr_enabled, gr_unproductive, gr_prev_modes, gr_used_last,
                          k_lost, n_stuck, n_active */
  /* read-only diagnostics written by the last unit */
  CHISAO_P = 20,       /* [N][d] last L-BFGS direction */
  CHISAO_LS_B = 21,    /* [N] i32 accepted trial index, -1 none accepted, -2 skipped */
  CHISAO_GHAT = 25,    /* [N][d] last HLC estimate */
  CHISAO_HLC_F = 26,   /* [N][M] last HLC values */
  CHISAO_RS_SRC = 27,  /* [N] i32 reseed source (RM: sample, GR: peak), -1 if not reseeded */
  CHISAO_RS_CAND = 28, /* [N] i32 RM: chosen candidate; GR: 2*column + sign */
  CHISAO_XT = 31,      /* [N][d] last line-search trial point */
  CHISAO_GR_Q = 32,    /* [d][d] last Golden-Rooster basis, element (r, c) at r*d + c */
  CHISAO_SIGMA = 33    /* [1] smoothing scale used by the last Hands-Like-Clouds step */
};

/* Units for chisao_phase (exactly one unit on the current state; used by teacher-forced parity tests). */
enum {
  CHISAO_PH_RELEASE_EVAL = 1,  /* release all + f, g at the current positions */
  CHISAO_PH_STICK = 2,         /* Eq. 3    */
  CHISAO_PH_DEDUP = 3,         /* Eq. 4 + index lists + Golden-Rooster bookkeeping   */
  CHISAO_PH_RESEED = 4,        /* Repulse Monkey / Golden Rooster / uniform refill  */
  CHISAO_PH_HLC_STEP = 5,      /* one Hands-Like-Clouds step `iter` (1-based)  */
  CHISAO_PH_ANTI_STEP = 6,     /* one momentum anti-convergence step `iter`  */
  CHISAO_PH_LBFGS_ITER = 11,   /* one L-BFGS iteration `iter` (1-based)    */
  CHISAO_PH_LBFGS_DIRECTION = 12 /* only the two-loop recursion + first trial point of an iteration (the HBM-bound
                                  history kernel; used by bench.py to time it with a full history)          */
};

/* Bytes of device workspace chisao_init needs for (cfg, obj).  Host only; no CUDA call. */
CHISAO_API int chisao_workspace_bytes(const chisao_config *cfg, const chisao_objective *obj, size_t *bytes);

/* Create a context.  x_dev: [N][d] fp32 population, read and written in place by every step.
 * workspace_dev: >= chisao_workspace_bytes, 256-byte aligned.  Enqueues parameter uploads and state
 * zeroing on `stream`; does not synchronise.  cycle = 0, Golden Rooster enabled. */
CHISAO_API int chisao_init(chisao_ctx **out, const chisao_config *cfg, const chisao_objective *obj,
                float *x_dev, void *workspace_dev, size_t workspace_bytes, void *stream);

/* x <- i.i.d. uniform in Theta from the Philox stream (Prop. 2 "uniform random"; R-15 tag INIT). */
CHISAO_API int chisao_seed_population(chisao_ctx *ctx);

/* ONE full oscillation cycle k = ++cycle (Alg. 1 body); phases 4-6 are skipped when
 * k == n_osc.  Asynchronous on the stream when stats == NULL; otherwise synchronises and
 * fills *stats.  Returns CHISAO_E_STATE once cycle == n_osc. */
CHISAO_API int chisao_step(chisao_ctx *ctx, chisao_stats *stats_or_null);

/* Host-buffer variant of chisao_step: copies x_host_in [N][d] to the device (if non-NULL), runs one cycle,
 * copies x, f and the stuck mask back to the given HOST buffers (each may be NULL) and synchronises. */
CHISAO_API int chisao_step_host(chisao_ctx *ctx, const float *x_host_in, float *x_host_out, float *f_host_out,
                     uint8_t *stuck_host_out, chisao_stats *stats_or_null);

/* "return {x_i : stuck_i}", sorted by (f descending, index ascending).  modes_out [cap][d],
 * f_out [cap], idx_out [cap] are HOST buffers (each may be NULL); *n_modes is always set; returns
 * CHISAO_E_CAPACITY (after filling the first cap rows) when cap < *n_modes.  Synchronises the stream. */
CHISAO_API int chisao_modes(chisao_ctx *ctx, float *modes_out, float *f_out, int32_t *idx_out, int32_t cap,
                 int32_t *n_modes);

/* State exchange through HOST buffers of exactly the field's size (else CHISAO_E_INVALID); synchronises. */
CHISAO_API int chisao_get_state(chisao_ctx *ctx, int32_t field, void *host_dst, size_t bytes);
CHISAO_API int chisao_set_state(chisao_ctx *ctx, int32_t field, const void *host_src, size_t bytes);

/* Test hook: run exactly one unit (CHISAO_PH_*) on the current state; `iter` is the 1-based iteration for
 * LBFGS_ITER / HLC_STEP / ANTI_STEP.  Does not advance the cycle counter.  Asynchronous. */
CHISAO_API int chisao_phase(chisao_ctx *ctx, int32_t phase_id, int32_t iter);

/* Fill *stats from the device control block (synchronises). */
CHISAO_API int chisao_get_stats(chisao_ctx *ctx, chisao_stats *stats);

/* Options outside the paper's parameter list.  CHISAO_OPT_STENCIL_AWARE (value 0 / 1, default 0): finite-difference
 * gradients of the dense objectives (GMM_FULL, QUAD) are computed by the stencil-aware evaluator, which shares
 * W (x - mu), |.|^2 and W^T W (x - mu) between the 2d stencil points of a sample (q(x +- h e_j) = q0 +- 2 h t_j +
 * h^2 cc_j).  It returns the same 2d values within rounding and counts
 * the same evaluations, but it is NOT a black-box evaluation of f: numbers obtained with it are
 * reported separately.  CHISAO_E_INVALID for other objectives or unknown options. */
#define CHISAO_OPT_STENCIL_AWARE 1
/* CHISAO_OPT_CUDA_GRAPH (default 1): chisao_step submits the cycle as ONE CUDA graph launch.  The launch sequence of a
 * cycle is static (every kernel reads its counts from the device control block); it is captured on an internal stream
 * that is forked from and joined to the caller's stream with events, and applied to the instantiated graph with
 * cudaGraphExecUpdate (the cycle index is a kernel argument).  Results are identical to direct submission; direct
 * submission is used while per-launch timing is enabled, by chisao_phase, and if the graph machinery fails. */
#define CHISAO_OPT_CUDA_GRAPH 2
/* CHISAO_OPT_LS_TILE_LOCAL (default: chosen at chisao_init from the cost of one evaluation tile): form of the
 * backtracking line search of an L-BFGS iteration (R-4 (iv)).  1: one launch runs every trial b = 0..ls_max -- a tile of
 * 256 searching samples repeats evaluate -> Armijo -> shrink until none of its samples retries; 0: one launch per trial
 * on worklists compacted between the trials (ls_max + 1 launches).  Per sample the arithmetic is the same (same
 * evaluator, noise slot, Armijo test, shrink), so the results are identical; 1 is the default for the FP32-FMA evaluators
 * of the small objectives and for QUAD / RFF on the tensor cores, 0 for the x-stationary GMM_FULL evaluator (a tile
 * streams the whole mixture: retries must stay dense), for which 1 returns CHISAO_E_INVALID. */
#define CHISAO_OPT_LS_TILE_LOCAL 3
/* CHISAO_OPT_LBFGS_RESIDENT (default: on where it exists): Phase 1 in its history-RESIDENT form -- one launch runs all
 * n_conv L-BFGS iterations (and, inside chisao_step, the release + first evaluation before them and Phase 2's partials after
 * them) for the samples a CTA keeps for the whole pass, with the (s, y) history in registers and never in HBM
 * (BASELINE.json north_star).  It exists for the FP32-FMA evaluators when d is 1, 2, 4, 8, 16 or 32, the
 * objective's parameters fit one shared-memory chunk and lbfgs_m <= 16 (C1, C2), else 1 returns CHISAO_E_INVALID; 0
 * selects the spill form (history in HBM, one group of launches per iteration), the only one at larger d or with the
 * tensor-core evaluators.  Both are checked against the oracle by the same teacher-forced tests. */
#define CHISAO_OPT_LBFGS_RESIDENT 4
CHISAO_API int chisao_set_option(chisao_ctx *ctx, int32_t option, int32_t value);

/* Which evaluator the context runs (decided at chisao_init from the objective, d and the value ranges):
 * CHISAO_INFO_EVALUATOR -> 0 FP32-FMA evaluator; 1 tensor cores, 3xTF32, A = x - c per component (QUAD at d > 32);
 * 2 tensor cores, x-stationary form with tf32 hi / lo operands; 3 the same with fp16 hi / lo operands (kind::f16; chosen
 * for GMM_FULL at d > 32 when max |W| and the box radius lie in [2^-3, 2^13]); 4 tensor cores,
 * random-Fourier phases w_j . x as an exact contraction of 10-bit fixed-point fp16 pieces (RFF at d <= 32, K <= 256
 * with max |w| and the box radius + 8 sigma_s + h in [2^-7, 2^10]; CHISAO_RFF_FP64 in the environment keeps the
 * FP32-FMA evaluator with fp64 phases); 5 tensor cores, QUAD at d > 32 with A = 2^k (x - c) per point and 2^ws W as fp16
 * hi / lo operands (kind::f16; the default for QUAD, CHISAO_TC_TF32 in the environment keeps form 1). */
#define CHISAO_INFO_EVALUATOR 1
#define CHISAO_INFO_GRAPH_LAUNCHES 2   /* cycles submitted as a CUDA graph so far */
#define CHISAO_INFO_LS_TILE_LOCAL 3    /* 1 if the line search runs every trial of a tile in one launch */
#define CHISAO_INFO_LBFGS_RESIDENT 4   /* 1 if Phase 1 runs in its history-resident form */
CHISAO_API int chisao_get_info(const chisao_ctx *ctx, int32_t which, int32_t *value);

/* Number of kernel launches this context has enqueued so far (host counter). */
CHISAO_API uint64_t chisao_launch_count(const chisao_ctx *ctx);

/* Device time in ms accumulated by the kernel class `which` since chisao_timing_reset, measured with CUDA
 * events on the context's stream when timing is enabled; also returns the launch count of that class.
 * chisao_timing_enable(ctx, on): on = 0 off, 1 every class, otherwise a mask with bit k + 1 selecting class k
 * (bracketing costs two event records per launch: measurable on the launch-bound configurations).
 * Classes: 0 eval_fd, 1 eval_points, 2 hlc, 3 lbfgs_direction, 4 lbfgs_update, 5 stick/dedup/lists,
 * 6 reseed.  chisao_timing_get synchronises. */
CHISAO_API int chisao_timing_enable(chisao_ctx *ctx, int32_t on);
CHISAO_API int chisao_timing_reset(chisao_ctx *ctx);
CHISAO_API int chisao_timing_get(chisao_ctx *ctx, int32_t which, double *ms, uint64_t *launches);

/* Pipe-rate probes for the roofline denominators (FP32 FMA and special-function rates are to be
 * measured in the same run, because the clocks under load differ from the nominal ones).  Runs a hand-written
 * micro-benchmark kernel (8 CTAs of 256 threads per SM, 8 independent dependency chains per thread) on `stream`, timed with
 * CUDA events, best of 5 after one warm-up; *value = TFLOP/s (CHISAO_PEAK_FP32_FMA: 2 flop per FFMA) or T operations/s
 * (CHISAO_PEAK_SFU: MUFU.EX2).  scratch_dev: >= 4 bytes of device memory.  Synchronises.  Not part of the CHISAO path. */
#define CHISAO_PEAK_FP32_FMA 0
#define CHISAO_PEAK_SFU 1
CHISAO_API int chisao_measure_peak(int32_t which, float *scratch_dev, void *stream, double *value);

/* Phase 2 of a cycle -- the stick test, Eq. 3 (Alg. 1 "f_max <- max_i f(x_i)", R-13) -- on the CALLER'S
 * arrays, for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): no context, no workspace, and the call makes NO cudaMalloc / cudaFree or other allocating call.
 *   stuck_i = (max_j |g_ij| < eps_grad) and f_i finite and (f_i >= f_max + log_delta),  f_max = max over the finite f_i
 * -- the same arithmetic, in the same precision, as CHISAO_PH_STICK of a context (a NaN in row i of g gives stuck_i = 0).
 * Arguments, all DEVICE pointers owned by the caller, on the current device:
 *   g_dev [N][d] fp32 row-major, f_dev [N] fp32 (read);  stuck_dev [N] u8 (written: 0 / 1);
 *   n_stuck_dev (may be NULL) int32: the number of stuck samples;  f_max_dev (may be NULL) fp32: f_max, -inf if no f_i is
 *   finite or N = 0.  0 <= N <= CHISAO_STATIC_MAX_N, 1 <= d <= CHISAO_MAX_D.
 * Asynchronous on `stream` (a cudaStream_t; NULL = the default stream); returns CHISAO_E_INVALID for N beyond
 * CHISAO_STATIC_MAX_N (or bad N, d, null pointers) and CHISAO_E_CUDA for runtime errors, with the text in
 * chisao_last_error(NULL).
 * Scratch: the per-sample ||grad f||_inf and the running f_max live in a file-scope device array of
 * CHISAO_STATIC_SCRATCH_BYTES (1 MiB + 256 bytes), which every GPU that loads the library holds until the process exits;
 * its device address is looked up on the first call on a device (cudaGetSymbolAddress -- make that first call outside a
 * stream capture).  Every call on a device shares the array and finds the previous call's contents in it: the call clears what
 * must start at zero on `stream` first.  Calls that OVERLAP on the GPU (different streams without a dependency between them)
 * race on it; calls on one stream, or ordered by events, are safe. */
#define CHISAO_STATIC_MAX_N 262144
#define CHISAO_STATIC_SCRATCH_BYTES (256 + 4 * CHISAO_STATIC_MAX_N)
CHISAO_API int chisao_stick_test_static(const float *g_dev, const float *f_dev, int32_t N, int32_t d, float eps_grad,
                                        float log_delta, uint8_t *stuck_dev, int32_t *n_stuck_dev, float *f_max_dev,
                                        void *stream);

CHISAO_API const char *chisao_last_error(const chisao_ctx *ctx_or_null);
CHISAO_API void chisao_destroy(chisao_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
