/* chisao_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of one CHISAO oscillation cycle, written from the paper
 * (arxiv/paper_2606_26164, /root/reference/PAPER.md) step by step in the paper's order:
 *   Algorithm 1, phases 1-6 (Eq. 2-6), Table 1.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may load it.
 * It shares no code, header or table with the CUDA path (paper_2606_26164_b200/csrc, include/chisao.h);
 * the structs below are restated here on purpose.
 *
 * Where the paper is silent the readings of DESIGN.md "Readings" (R-1 ... R-17) are followed; each
 * function in chisao_oracle.c cites the passage or reading it implements.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): objective values vs scipy logsumexp /
 * multivariate_normal, FD gradients vs analytic gradients, two-loop recursion vs the dense BFGS
 * inverse update, L-BFGS vs the exact maximiser of a quadratic, Eq. 3 / Eq. 4 / Eq. 6 brute force and
 * closed forms, Eq. 9 unbiasedness, Remark 1, d=2 grid mode enumeration, Philox vs cuRAND's host
 * generator.  PARITY UNPINNED AGAINST THE PAPER (pinned GPU<->oracle only): the particular choices of
 * readings R-4 (line search details), R-8 (Repulse Monkey details), R-9 (Golden Rooster details) and
 * R-12 (step sizes) -- the paper prints no values that could check them.
 */
#ifndef CHISAO_ORACLE_H
#define CHISAO_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t id, d, K;
  const float *means, *mats, *vec_a, *vec_b;
  float scalar0, sigma_noise;
} orc_objective;

typedef struct {
  int32_t d, N;
  const float *lo, *hi;
  int32_t n_osc, n_conv, n_anti, n_cloud, hlc_M, lbfgs_m, ls_max, reseed_cands;
  float fd_h, eps_grad, eps_dup, log_delta, mu, alpha_anti, eta_hlc, sigma_s, ls_c1, ls_shrink;
  int32_t hlc_baseline;
  uint32_t phase_mask;
  uint64_t seed;
} orc_config;

typedef struct {
  int32_t cycle, n_stuck, k_lost, n_active, reseed_strategy, gr_enabled;
  uint64_t evals[8];
  double f_max;
} orc_stats;

typedef struct orc_ctx orc_ctx;

/* state fields for orc_get / orc_set (all exchanged as double unless noted) */
enum {
  ORC_X = 0, ORC_F = 1, ORC_G = 2, ORC_V = 3, ORC_STUCK = 4 /*u8*/, ORC_REMOVED = 5 /*u8*/,
  ORC_HIST_S = 6 /*[m][N][d], slot 0 = oldest*/, ORC_HIST_Y = 7, ORC_HIST_LEN = 8 /*i32*/,
  ORC_STALLED = 9 /*u8*/, ORC_CTRL = 10 /*i32[8]: cycle, gr_enabled, gr_unproductive, gr_prev_modes,
  gr_used_last, k_lost, n_stuck, n_active*/,
  /* diagnostics written by the last unit */
  ORC_P = 20, ORC_LS_B = 21 /*i32: accepted trial, -1 none accepted, -2 skipped*/, ORC_LS_MARGIN = 22,
  ORC_ASC_MARGIN = 23, ORC_CURV_MARGIN = 24, ORC_GHAT = 25, ORC_HLC_F = 26 /*[N][M]*/,
  ORC_RS_SRC = 27 /*i32*/, ORC_RS_CAND = 28 /*i32*/, ORC_RS_MARGIN = 29, ORC_HLC_U = 30 /*[N][M][d]*/,
  ORC_SIGMA = 33 /*double[1]: smoothing scale used by the last HLC step*/,
  ORC_RS_SCORE = 34 /*[N][16]: Repulse Monkey, score (min squared L2 distance to the frozen modes) of candidate c of a slot*/
};

/* units for orc_phase */
enum { ORC_PH_RELEASE_EVAL = 1, ORC_PH_STICK = 2, ORC_PH_DEDUP = 3, ORC_PH_RESEED = 4,
       ORC_PH_HLC_STEP = 5, ORC_PH_ANTI_STEP = 6, ORC_PH_LBFGS_ITER = 11 };

orc_ctx *orc_create(const orc_config *cfg, const orc_objective *obj, const float *x0);
void orc_destroy(orc_ctx *);
void orc_set_threads(orc_ctx *, int nthreads);      /* outer loop over samples only */
int  orc_step(orc_ctx *, orc_stats *out);           /* one full cycle k = ++cycle */
int  orc_phase(orc_ctx *, int phase_id, int iter);  /* exactly one unit on the current state */
int  orc_modes(orc_ctx *, double *modes, double *f, int32_t *idx, int32_t cap, int32_t *n_modes);
int  orc_get(orc_ctx *, int field, void *dst, uint64_t bytes);
int  orc_set(orc_ctx *, int field, const void *src, uint64_t bytes);
void orc_stats_now(orc_ctx *, orc_stats *out);

/* pure helpers exposed so tests can pin them one by one */
void   orc_objective_values(orc_ctx *, const double *pts, int64_t npts, double *f_out); /* noise-free */
void   orc_fd_gradient(orc_ctx *, const double *x, double *f_out, double *g_out);       /* noise-free */
void   orc_two_loop(int d, int len, const double *S, const double *Y, const double *gamma, double *r);
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_uniform(uint64_t seed, uint32_t c1, uint32_t c2, uint32_t c3, uint64_t n);
double orc_normal(uint64_t seed, uint32_t c1, uint32_t c2, uint32_t c3, uint64_t n);
void   orc_gr_basis(orc_ctx *, int cycle, double *Q /*[d][d], column c = Q[r*d+c]*/);
double orc_noise(orc_ctx *, int cycle, int sample, int phase, int iter, int slot);

#ifdef __cplusplus
}
#endif
#endif
