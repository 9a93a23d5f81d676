/* chisao_oracle.c -- TEST INFRASTRUCTURE (see chisao_oracle.h): fp64 CPU oracle of the CHISAO cycle.
 *
 * Every function cites the passage of /root/reference/PAPER.md (or the DESIGN.md reading R-n) it
 * follows.  Plain loops, one sample at a time, no blocking, no fusion; the only parallelism is an
 * optional OpenMP `for` over the sample index ("every operation vectorizes over i").
 * Positions (x, v) are rounded to fp32 after every update so that both sides of a teacher-forced
 * parity check start every unit from bit-identical inputs.
 */
#include "chisao_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { PUR_INIT = 0, PUR_NOISE = 1, PUR_HLC_U = 2, PUR_RS_SRC = 3, PUR_RS_T = 4, PUR_RS_DIR = 5,
       PUR_GR_MATRIX = 6, PUR_RS_UNIF = 7 };
enum { EV_INIT = 0, EV_LS = 1, EV_LBFGS_FD = 2, EV_HLC = 5, EV_ANTI = 6 };

struct orc_ctx {
  orc_config c;
  orc_objective o;
  int nthreads;
  double *lo, *hi;
  /* objective parameters promoted to fp64 from the SAME fp32 arrays the CUDA path receives */
  double *means, *mats, *va, *vb;
  double s0, sigma_noise;
  /* state */
  double *x, *f, *g, *v, *S, *Y;      /* S,Y: [N][m][d], slot 0 = oldest */
  int32_t *len;
  uint8_t *stuck, *removed, *stalled;
  int32_t cycle, gr_enabled, gr_unproductive, gr_prev_modes, gr_used_last;
  int32_t k_lost, n_stuck, n_active, reseed_strategy;
  double f_max, sigma_eff;
  uint64_t evals[8];
  /* diagnostics */
  double *p, *ls_margin, *asc_margin, *curv_margin, *ghat, *hlc_f, *hlc_u, *rs_margin;
  int32_t *ls_b, *rs_src, *rs_cand;
  double *rs_score;                  /* [N][16] diagnostic: the score (min squared distance to the modes) of every candidate */
};

/* ------------------------------------------------------------------------------------------------
 * Counter-based randomness: Philox4x32-10 (Salmon et al., SC'11), reading R-15.
 * The paper never says how it draws; BASELINE.json north_star fixes "a counter-based Philox stream
 * keyed by (seed, cycle, sample, draw)".
 * ---------------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void philox_block(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t w[4]) {
  uint32_t ctr[4] = { c0, c1, c2, c3 }, key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
  orc_philox4x32_10(ctr, key, w);
}
static uint32_t tag(int phase, int iter, int purpose) {
  return ((uint32_t)phase << 24) | ((uint32_t)(iter & 0xFFFF) << 8) | (uint32_t)purpose;
}
/* word -> uniform in (0,1): u = ((w >> 9) + 0.5) 2^-23 = (2k+1)/2^24 with k < 2^23, which is exact in
 * fp32 as well as fp64 (R-15; a 24-bit k would need 25 significant bits) */
static double u01(uint32_t w) { return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0); }

/* n-th uniform of the sequence (c1,c2,c3): word n mod 4 of block n div 4 (R-15) */
double orc_uniform(uint64_t seed, uint32_t c1, uint32_t c2, uint32_t c3, uint64_t n) {
  uint32_t w[4];
  philox_block(seed, (uint32_t)(n / 4), c1, c2, c3, w);
  return u01(w[n % 4]);
}
/* n-th normal: Box-Muller on (w0,w1) -> lanes 0,1 and (w2,w3) -> lanes 2,3 of block n div 4 (R-15) */
double orc_normal(uint64_t seed, uint32_t c1, uint32_t c2, uint32_t c3, uint64_t n) {
  uint32_t w[4];
  philox_block(seed, (uint32_t)(n / 4), c1, c2, c3, w);
  int lane = (int)(n % 4), pair = lane / 2;
  double u1 = u01(w[2 * pair]), u2 = u01(w[2 * pair + 1]);
  double r = sqrt(-2.0 * log(u1)), a = 2.0 * M_PI * u2;
  return (lane % 2 == 0) ? r * cos(a) : r * sin(a);
}
/* additive evaluation noise eps ~ N(0, sigma_noise^2); one independent draw per
 * evaluation keyed structurally by (cycle, sample, phase, iteration, slot) (R-2) */
double orc_noise(orc_ctx *s, int cycle, int sample, int phase, int iter, int slot) {
  if (s->sigma_noise == 0.0) return 0.0;
  uint32_t w[4];
  philox_block(s->c.seed, (uint32_t)slot, (uint32_t)sample, (uint32_t)cycle, tag(phase, iter, PUR_NOISE), w);
  double u1 = u01(w[0]), u2 = u01(w[1]);
  return s->sigma_noise * sqrt(-2.0 * log(u1)) * cos(2.0 * M_PI * u2);
}

/* ------------------------------------------------------------------------------------------------
 * Objectives (value only: "accessible through evaluations f(theta)").
 * ---------------------------------------------------------------------------------------------- */
static double logsumexp(const double *v, int n) {
  double m = v[0];
  for (int k = 1; k < n; ++k) if (v[k] > m) m = v[k];
  if (!isfinite(m)) return m;
  double acc = 0.0;
  for (int k = 0; k < n; ++k) acc += exp(v[k] - m);
  return m + log(acc);
}

static double objective(const orc_ctx *s, const double *x) {
  const int d = s->o.d, K = s->o.K;
  switch (s->o.id) {
  case 0: { /* log sum_k w_k N(x; mu_k, sigma^2 I), PAPER.md:629 (App. D "Gaussian mixture") */
    double sig = s->mats[0];
    double *v = (double *)alloca(sizeof(double) * K);
    for (int k = 0; k < K; ++k) {
      double r2 = 0.0;
      for (int j = 0; j < d; ++j) { double t = x[j] - s->means[k * d + j]; r2 += t * t; }
      v[k] = s->va[k] - r2 / (2.0 * sig * sig);
    }
    return logsumexp(v, K);
  }
  case 1: { /* diagonal-covariance mixture (BASELINE.json configs[1]) */
    double *v = (double *)alloca(sizeof(double) * K);
    for (int k = 0; k < K; ++k) {
      double q = 0.0;
      for (int j = 0; j < d; ++j) { double t = (x[j] - s->means[k * d + j]) * s->mats[k * d + j]; q += t * t; }
      v[k] = s->va[k] - 0.5 * q;
    }
    return logsumexp(v, K);
  }
  case 2: { /* full-covariance mixture, Sigma_k^-1 = W_k^T W_k (BASELINE.json configs[4]) */
    double *v = (double *)alloca(sizeof(double) * K);
    for (int k = 0; k < K; ++k) {
      const double *W = s->mats + (size_t)k * d * d;
      double q = 0.0;
      for (int r = 0; r < d; ++r) {
        double z = 0.0;
        for (int c = 0; c < d; ++c) z += W[r * d + c] * (x[c] - s->means[k * d + c]);
        q += z * z;
      }
      v[k] = s->va[k] - 0.5 * q;
    }
    return logsumexp(v, K);
  }
  case 3: { /* f = -||x||^2/50 + sum_j a_j cos(w_j.x + b_j) (BASELINE.json configs[2]) */
    double n2 = 0.0, acc = 0.0;
    for (int j = 0; j < d; ++j) n2 += x[j] * x[j];
    for (int k = 0; k < K; ++k) {
      double t = s->vb[k];
      for (int j = 0; j < d; ++j) t += s->mats[k * d + j] * x[j];
      acc += s->va[k] * cos(t);
    }
    return -s->s0 * n2 + acc;
  }
  case 4: { /* f = -1/2 (x-c)^T Q^T diag(lambda) Q (x-c) = -1/2 ||W (x-c)||^2 (BASELINE.json configs[3]) */
    double q = 0.0;
    for (int r = 0; r < d; ++r) {
      double z = 0.0;
      for (int c = 0; c < d; ++c) z += s->mats[r * d + c] * (x[c] - s->means[c]);
      q += z * z;
    }
    return -0.5 * q;
  }
  /* Appendix D of the paper, "Benchmark Function Definitions", all negated for maximisation */
  case 5: { /* Rastrigin: f = -[A d + sum (x_i^2 - A cos(2 pi x_i))], A = 10 */
    double acc = 10.0 * d;
    for (int j = 0; j < d; ++j) acc += x[j] * x[j] - 10.0 * cos(2.0 * M_PI * x[j]);
    return -acc;
  }
  case 6: { /* Ackley: a = 20, b = 0.2, c = 2 pi */
    double s2 = 0.0, sc = 0.0;
    for (int j = 0; j < d; ++j) { s2 += x[j] * x[j]; sc += cos(2.0 * M_PI * x[j]); }
    return -(-20.0 * exp(-0.2 * sqrt(s2 / d)) - exp(sc / d) + 20.0 + M_E);
  }
  case 7: { /* Schwefel: f = -[418.9829 d - sum x_i sin(sqrt|x_i|)] */
    double acc = 0.0;
    for (int j = 0; j < d; ++j) acc += x[j] * sin(sqrt(fabs(x[j])));
    return -(418.9829 * d - acc);
  }
  case 8: { /* Styblinski-Tang: f = -1/2 sum (x^4 - 16 x^2 + 5 x) */
    double acc = 0.0;
    for (int j = 0; j < d; ++j) { double t = x[j]; acc += t * t * t * t - 16.0 * t * t + 5.0 * t; }
    return -0.5 * acc;
  }
  case 9: { /* Michalewicz: f = sum sin(x_i) sin^{2m}(i x_i^2 / pi), m = 10, i = 1..d */
    double acc = 0.0;
    for (int j = 0; j < d; ++j) acc += sin(x[j]) * pow(sin((j + 1) * x[j] * x[j] / M_PI), 20.0);
    return acc;
  }
  case 10: { /* Trid: f = -[sum (x_i - 1)^2 - sum_{i>=2} x_i x_{i-1}] */
    double acc = 0.0;
    for (int j = 0; j < d; ++j) acc += (x[j] - 1.0) * (x[j] - 1.0);
    for (int j = 1; j < d; ++j) acc -= x[j] * x[j - 1];
    return -acc;
  }
  case 11: { /* Bukin N.6, PAPER.md:627 (d = 2): f = -[100 sqrt|y - 0.01 x^2| + 0.01 |x + 10|] */
    return -(100.0 * sqrt(fabs(x[1] - 0.01 * x[0] * x[0])) + 0.01 * fabs(x[0] + 10.0));
  }
  }
  return NAN;
}

void orc_objective_values(orc_ctx *s, const double *pts, int64_t npts, double *f_out) {
  for (int64_t i = 0; i < npts; ++i) f_out[i] = objective(s, pts + i * s->o.d);
}

/* Central finite differences (PAPER.md:62 "computed by finite differences", :555 "2dN finite-difference
 * evaluations per L-BFGS step"; R-1: central, absolute step h, stencil points not clipped).
 * Evaluation slots: 0 = centre, 1+2j = x + h e_j, 2+2j = x - h e_j (R-2). */
static void eval_fd(orc_ctx *s, int i, const double *x, int phase, int iter, int with_centre,
                    double *f_out, double *g_out, int counter) {
  const int d = s->c.d;
  const double h = (double)s->c.fd_h;
  double *xp = (double *)alloca(sizeof(double) * d);
  if (with_centre) {
    *f_out = objective(s, x) + orc_noise(s, s->cycle, i, phase, iter, 0);
  }
  for (int j = 0; j < d; ++j) {
    memcpy(xp, x, sizeof(double) * d);
    xp[j] = x[j] + h;
    double fp = objective(s, xp) + orc_noise(s, s->cycle, i, phase, iter, 1 + 2 * j);
    xp[j] = x[j] - h;
    double fm = objective(s, xp) + orc_noise(s, s->cycle, i, phase, iter, 2 + 2 * j);
    g_out[j] = (fp - fm) / (2.0 * h);
  }
  if (counter >= 0) {
#pragma omp atomic
    s->evals[counter] += (uint64_t)(2 * d + (with_centre ? 1 : 0));
  }
}

void orc_fd_gradient(orc_ctx *s, const double *x, double *f_out, double *g_out) {
  double sn = s->sigma_noise;
  s->sigma_noise = 0.0;
  eval_fd(s, 0, x, 0, 0, 1, f_out, g_out, -1);
  s->sigma_noise = sn;
}

static double clipf32(double v, double lo, double hi) {
  if (v < lo) v = lo;
  if (v > hi) v = hi;
  return (double)(float)v; /* positions are fp32 state (north_star "N fp32"); see file header */
}

/* ------------------------------------------------------------------------------------------------
 * Phase 1 (Eq. 2; Alg. 1 lines "stuck <- False^N", "x, grad f <- L-BFGS_batch").
 * ---------------------------------------------------------------------------------------------- */

/* O-1: release all + first evaluation f, g at the current positions */
static void phase_release_eval(orc_ctx *s) {
  const int N = s->c.N, d = s->c.d;
#pragma omp parallel for schedule(dynamic, 16) num_threads(s->nthreads)
  for (int i = 0; i < N; ++i) {
    s->stuck[i] = 0; s->removed[i] = 0; s->stalled[i] = 0; s->len[i] = 0; /* history reset: R-5 */
    eval_fd(s, i, s->x + (size_t)i * d, 1, 0, 1, &s->f[i], s->g + (size_t)i * d, EV_INIT);
  }
}

/* L-BFGS two-loop recursion (Nocedal & Wright Alg. 7.4 = refs [19,20] of PAPER.md:77), memory m
 * (PAPER.md:82).  S, Y: [len][d], slot 0 = oldest.  Returns r = H_k gamma with
 * H_0 = (s.y / y.y) I of the newest pair (R-4). */
void orc_two_loop(int d, int len, const double *S, const double *Y, const double *gamma, double *r) {
  double alpha[64], rho[64];
  for (int j = 0; j < d; ++j) r[j] = gamma[j];
  for (int l = len - 1; l >= 0; --l) {
    double sy = 0.0, sq = 0.0;
    for (int j = 0; j < d; ++j) { sy += S[l * d + j] * Y[l * d + j]; sq += S[l * d + j] * r[j]; }
    rho[l] = 1.0 / sy;
    alpha[l] = rho[l] * sq;
    for (int j = 0; j < d; ++j) r[j] -= alpha[l] * Y[l * d + j];
  }
  if (len > 0) {
    double sy = 0.0, yy = 0.0;
    const double *sn = S + (len - 1) * d, *yn = Y + (len - 1) * d;
    for (int j = 0; j < d; ++j) { sy += sn[j] * yn[j]; yy += yn[j] * yn[j]; }
    for (int j = 0; j < d; ++j) r[j] *= sy / yy;
  }
  for (int l = 0; l < len; ++l) {
    double yr = 0.0;
    for (int j = 0; j < d; ++j) yr += Y[l * d + j] * r[j];
    double beta = rho[l] * yr;
    for (int j = 0; j < d; ++j) r[j] += S[l * d + j] * (alpha[l] - beta);
  }
}

/* O-2: one L-BFGS iteration for sample i; maximise f <=> minimise phi = -f, gamma = -g (R-4). */
static void lbfgs_iter_sample(orc_ctx *s, int i, int it) {
  const int d = s->c.d, m = s->c.lbfgs_m;
  double *x = s->x + (size_t)i * d, *g = s->g + (size_t)i * d, *p = s->p + (size_t)i * d;
  double *S = s->S + (size_t)i * m * d, *Y = s->Y + (size_t)i * m * d;
  double *gam = (double *)alloca(sizeof(double) * d), *xt = (double *)alloca(sizeof(double) * d);
  double *gn = (double *)alloca(sizeof(double) * d), *r = (double *)alloca(sizeof(double) * d);
  s->ls_b[i] = -2; s->ls_margin[i] = INFINITY; s->asc_margin[i] = INFINITY; s->curv_margin[i] = INFINITY;
  for (int j = 0; j < d; ++j) p[j] = 0.0;
  /* (i) already stationary (Eq. 3's gradient test) or stalled: nothing to do, no evaluations (R-6) */
  double ginf = 0.0;
  for (int j = 0; j < d; ++j) if (fabs(g[j]) > ginf) ginf = fabs(g[j]);
  if (s->stalled[i] || !(ginf >= (double)s->c.eps_grad)) return;
  double gnorm2 = 0.0;
  for (int j = 0; j < d; ++j) { gam[j] = -g[j]; gnorm2 += g[j] * g[j]; }
  /* (ii) direction */
  if (s->len[i] > 0) {
    orc_two_loop(d, s->len[i], S, Y, gam, r);
    double gp = 0.0, pn2 = 0.0;
    for (int j = 0; j < d; ++j) { p[j] = -r[j]; gp += gam[j] * p[j]; pn2 += p[j] * p[j]; }
    s->asc_margin[i] = fabs(gp) / (sqrt(gnorm2 * pn2) + 1e-300);
    if (!(gp < 0.0)) { /* not a descent direction for phi: steepest restart, clear history */
      for (int j = 0; j < d; ++j) p[j] = -gam[j];
      s->len[i] = 0;
    }
  } else {
    for (int j = 0; j < d; ++j) p[j] = -gam[j];
  }
  /* (iii) first trial step */
  double t0 = (s->len[i] > 0) ? 1.0 : fmin(1.0, 1.0 / sqrt(gnorm2));
  /* (iv) backtracking Armijo on projected trial points */
  const double phi = -s->f[i];
  int acc = -1; double phit = 0.0, t = t0;
  for (int b = 0; b <= s->c.ls_max; ++b, t *= (double)s->c.ls_shrink) {
    double dec = 0.0;
    for (int j = 0; j < d; ++j) {
      xt[j] = clipf32(x[j] + t * p[j], s->lo[j], s->hi[j]);
      dec += gam[j] * (xt[j] - x[j]);
    }
    phit = -(objective(s, xt) + orc_noise(s, s->cycle, i, 1, it, 2 * d + 1 + b));
#pragma omp atomic
    s->evals[EV_LS] += 1;
    double rhs = phi + (double)s->c.ls_c1 * dec;
    double scale = fmax(fmax(fabs(phit), fabs(phi)), 1.0);
    double mg = fabs(phit - rhs) / scale;
    if (mg < s->ls_margin[i]) s->ls_margin[i] = mg;
    if (isfinite(phit) && phit <= rhs) { acc = b; break; }
  }
  s->ls_b[i] = acc;
  if (acc < 0) { /* (v) no trial accepted */
    if (s->len[i] == 0) s->stalled[i] = 1; else s->len[i] = 0;
    return;
  }
  /* (vi) accepted: gradient at the new point (2d evaluations), curvature pair */
  double fdummy;
  eval_fd(s, i, xt, 1, it, 0, &fdummy, gn, EV_LBFGS_FD);
  double sy = 0.0, ss = 0.0, yy = 0.0;
  double *sv = r, *yv = gam; /* reuse */
  for (int j = 0; j < d; ++j) {
    sv[j] = xt[j] - x[j];
    yv[j] = (-gn[j]) - (-g[j]);
    sy += sv[j] * yv[j]; ss += sv[j] * sv[j]; yy += yv[j] * yv[j];
  }
  double thr = 1e-10 * sqrt(ss) * sqrt(yy);
  s->curv_margin[i] = fabs(sy - thr) / (sqrt(ss) * sqrt(yy) + 1e-300);
  if (sy > thr) {
    if (s->len[i] == m) { /* drop the oldest */
      memmove(S, S + d, sizeof(double) * (size_t)(m - 1) * d);
      memmove(Y, Y + d, sizeof(double) * (size_t)(m - 1) * d);
      s->len[i] = m - 1;
    }
    memcpy(S + (size_t)s->len[i] * d, sv, sizeof(double) * d);
    memcpy(Y + (size_t)s->len[i] * d, yv, sizeof(double) * d);
    s->len[i] += 1;
  }
  for (int j = 0; j < d; ++j) { x[j] = xt[j]; g[j] = gn[j]; }
  s->f[i] = -phit;
}

static void phase_lbfgs_iter(orc_ctx *s, int it) {
  const int N = s->c.N;
#pragma omp parallel for schedule(dynamic, 8) num_threads(s->nthreads)
  for (int i = 0; i < N; ++i) lbfgs_iter_sample(s, i, it);
}

/* ------------------------------------------------------------------------------------------------
 * Phase 2: stick detection, Eq. 3 with f_max = max_i f(x_i) (Alg. 1; R-13).
 * ---------------------------------------------------------------------------------------------- */
static void phase_stick(orc_ctx *s) {
  const int N = s->c.N, d = s->c.d;
  double fmax = -INFINITY;
  for (int i = 0; i < N; ++i) if (isfinite(s->f[i]) && s->f[i] > fmax) fmax = s->f[i];
  s->f_max = fmax;
  int ns = 0;
  for (int i = 0; i < N; ++i) {
    double ginf = 0.0;
    const double *g = s->g + (size_t)i * d;
    for (int j = 0; j < d; ++j) { double a = fabs(g[j]); if (!(a <= ginf)) ginf = a; } /* NaN -> NaN */
    s->stuck[i] = (ginf < (double)s->c.eps_grad) && isfinite(s->f[i]) &&
                  (s->f[i] >= fmax + (double)s->c.log_delta);
    s->removed[i] = 0;
    ns += s->stuck[i];
  }
  s->n_stuck = ns; s->k_lost = 0; s->n_active = N - ns;
}

/* ------------------------------------------------------------------------------------------------
 * Phase 3: L-infinity deduplication, Eq. 4 (Eq. 4 is garbled in the extraction --
 * reading R-7: "the sample with the higher function value survives", ties -> lower index survives,
 * every test against the pre-removal stuck set).
 * ---------------------------------------------------------------------------------------------- */
static void phase_dedup(orc_ctx *s) {
  const int N = s->c.N, d = s->c.d;
  const double eps = (double)s->c.eps_dup;
  if (s->c.phase_mask & (1u << 3)) {
#pragma omp parallel for schedule(dynamic, 64) num_threads(s->nthreads)
    for (int i = 0; i < N; ++i) {
      if (!s->stuck[i]) continue;
      int rem = 0;
      for (int j = 0; j < N && !rem; ++j) {
        if (j == i || !s->stuck[j]) continue;
        double dist = 0.0;
        for (int c = 0; c < d; ++c) {
          double a = fabs(s->x[(size_t)i * d + c] - s->x[(size_t)j * d + c]);
          if (a > dist) dist = a;
        }
        if (dist < eps && (s->f[j] > s->f[i] || (s->f[j] == s->f[i] && j < i))) rem = 1;
      }
      s->removed[i] = (uint8_t)rem;
    }
  }
  int kl = 0, ns = 0, na = 0;
  for (int i = 0; i < N; ++i) {
    if (s->removed[i]) { s->stuck[i] = 0; ++kl; }
    ns += s->stuck[i];
    na += (!s->stuck[i] && !s->removed[i]);
  }
  s->k_lost = kl; s->n_stuck = ns; s->n_active = na;
  /* Golden Rooster self-disable ("adaptively disables itself if successive generations
   * discover no new peaks"; R-9: two consecutive GR cycles with no increase of the mode count) */
  if (s->gr_used_last) {
    if (ns > s->gr_prev_modes) s->gr_unproductive = 0; else s->gr_unproductive += 1;
    if (s->gr_unproductive >= 2) s->gr_enabled = 0;
  }
}

/* ------------------------------------------------------------------------------------------------
 * Phase 4: reseeding.
 * ---------------------------------------------------------------------------------------------- */

/* distance along unit direction u from x to the boundary of the box Theta (one-sided ray) */
static double ray_exit(const orc_ctx *s, const double *x, const double *u) {
  double tmax = INFINITY;
  for (int j = 0; j < s->c.d; ++j) {
    double t = INFINITY;
    if (u[j] > 0.0) t = (s->hi[j] - x[j]) / u[j];
    else if (u[j] < 0.0) t = (s->lo[j] - x[j]) / u[j];
    if (t < tmax) tmax = t;
  }
  if (!(tmax >= 0.0) || !isfinite(tmax)) tmax = 0.0;
  return tmax;
}

/* Golden Rooster directions: QR of a random Gaussian matrix by modified Gram-Schmidt
 * with one re-orthogonalisation pass, R_ii > 0 (R-9).  Column c of Q is Q[r*d + c]. */
void orc_gr_basis(orc_ctx *s, int cycle, double *Q) {
  const int d = s->c.d;
  for (int a = 0; a < d; ++a)
    for (int b = 0; b < d; ++b)
      Q[a * d + b] = orc_normal(s->c.seed, 0u, (uint32_t)cycle, tag(4, 0, PUR_GR_MATRIX), (uint64_t)a * d + b);
  for (int c = 0; c < d; ++c) {
    for (int pass = 0; pass < 2; ++pass)
      for (int e = 0; e < c; ++e) {
        double dot = 0.0;
        for (int r = 0; r < d; ++r) dot += Q[r * d + e] * Q[r * d + c];
        for (int r = 0; r < d; ++r) Q[r * d + c] -= dot * Q[r * d + e];
      }
    double n2 = 0.0;
    for (int r = 0; r < d; ++r) n2 += Q[r * d + c] * Q[r * d + c];
    double inv = 1.0 / sqrt(n2);
    for (int r = 0; r < d; ++r) Q[r * d + c] *= inv;
  }
}

/* Repulse Monkey for one removed slot r (R-8) */
static void rm_slot(orc_ctx *s, int r, const int *A, int nA, const int *P, int nP, double *out) {
  const int d = s->c.d, C = s->c.reseed_cands;
  uint32_t w[4];
  philox_block(s->c.seed, 0u, (uint32_t)r, (uint32_t)s->cycle, tag(4, 0, PUR_RS_SRC), w);
  int src = A[(int)(((uint64_t)w[0] * (uint64_t)nA) >> 32)];
  double *u = (double *)alloca(sizeof(double) * d), *cand = (double *)alloca(sizeof(double) * d);
  double n2 = 0.0;
  for (int j = 0; j < d; ++j) {
    u[j] = orc_normal(s->c.seed, (uint32_t)r, (uint32_t)s->cycle, tag(4, 0, PUR_RS_DIR), (uint64_t)j);
    n2 += u[j] * u[j];
  }
  for (int j = 0; j < d; ++j) u[j] /= sqrt(n2);
  const double *xs = s->x + (size_t)src * d;
  double tmax = ray_exit(s, xs, u);
  double best = -1.0, second = -1.0; int bestc = 0;
  for (int c = 0; c < C; ++c) {
    double U = orc_uniform(s->c.seed, (uint32_t)r, (uint32_t)s->cycle, tag(4, 0, PUR_RS_T), (uint64_t)c);
    for (int j = 0; j < d; ++j) cand[j] = clipf32(xs[j] + tmax * U * u[j], s->lo[j], s->hi[j]);
    double mind = INFINITY;
    for (int pi = 0; pi < nP; ++pi) {
      const double *xp = s->x + (size_t)P[pi] * d;
      double d2 = 0.0;
      for (int j = 0; j < d; ++j) { double t = cand[j] - xp[j]; d2 += t * t; }
      if (d2 < mind) mind = d2;
    }
    if (c < 16) s->rs_score[(size_t)r * 16 + c] = mind;
    if (mind > best) { second = best; best = mind; bestc = c; memcpy(out, cand, sizeof(double) * d); }
    else if (mind > second) second = mind;
  }
  s->rs_src[r] = src; s->rs_cand[r] = bestc;
  s->rs_margin[r] = (isfinite(best) && best > 0.0) ? (best - second) / best : INFINITY;
}

static void phase_reseed(orc_ctx *s) {
  const int N = s->c.N, d = s->c.d;
  s->reseed_strategy = 0;
  s->gr_used_last = 0;
  for (int i = 0; i < N; ++i) { s->rs_src[i] = -1; s->rs_cand[i] = -1; s->rs_margin[i] = INFINITY; }
  if (s->k_lost <= 0 || !(s->c.phase_mask & (1u << 4))) return;
  int *A = (int *)malloc(sizeof(int) * N), *P = (int *)malloc(sizeof(int) * N), *R = (int *)malloc(sizeof(int) * N);
  int nA = 0, nP = 0, nR = 0;
  for (int i = 0; i < N; ++i) {          /* ascending index lists (R-10: unfrozen = not stuck, not removed) */
    if (s->removed[i]) R[nR++] = i; else if (s->stuck[i]) P[nP++] = i; else A[nA++] = i;
  }
  double *newx = (double *)malloc(sizeof(double) * (size_t)nR * d);
  if (nA >= 5) {
    /* Repulse Monkey: rays from unfrozen samples in random directions, uniform along
     * the ray within Theta; R-8: best of C candidates by distance to the frozen-mode set */
    s->reseed_strategy = 1;
#pragma omp parallel for schedule(dynamic, 16) num_threads(s->nthreads)
    for (int q = 0; q < nR; ++q) rm_slot(s, R[q], A, nA, P, nP, newx + (size_t)q * d);
  } else if (s->gr_enabled && nP > 0) {
    /* Golden Rooster: rays from confirmed peaks along orthonormal directions */
    s->reseed_strategy = 2;
    s->gr_used_last = 1; s->gr_prev_modes = nP;
    double *Q = (double *)malloc(sizeof(double) * d * d), *u = (double *)malloc(sizeof(double) * d);
    orc_gr_basis(s, s->cycle, Q);
    for (int q = 0; q < nR; ++q) {
      int r = R[q];
      int peak = P[q % nP], col = (q / nP) % d, neg = (int)(((int64_t)q / ((int64_t)nP * d)) % 2);
      for (int j = 0; j < d; ++j) u[j] = neg ? -Q[j * d + col] : Q[j * d + col];
      const double *xs = s->x + (size_t)peak * d;
      double tmax = ray_exit(s, xs, u);
      double U = orc_uniform(s->c.seed, (uint32_t)r, (uint32_t)s->cycle, tag(4, 0, PUR_RS_T), 0);
      for (int j = 0; j < d; ++j) newx[(size_t)q * d + j] = clipf32(xs[j] + tmax * U * u[j], s->lo[j], s->hi[j]);
      s->rs_src[r] = peak; s->rs_cand[r] = col * 2 + neg;
    }
    free(Q); free(u);
  } else {
    /* population is maintained at size N: uniform refill of Theta (R-9) */
    s->reseed_strategy = 3;
    for (int q = 0; q < nR; ++q) {
      int r = R[q];
      for (int j = 0; j < d; ++j) {
        double U = orc_uniform(s->c.seed, (uint32_t)r, (uint32_t)s->cycle, tag(4, 0, PUR_RS_UNIF), (uint64_t)j);
        newx[(size_t)q * d + j] = clipf32(s->lo[j] + U * (s->hi[j] - s->lo[j]), s->lo[j], s->hi[j]);
      }
    }
  }
  for (int q = 0; q < nR; ++q) { /* "All reseeded samples are marked as unstuck" */
    int r = R[q];
    memcpy(s->x + (size_t)r * d, newx + (size_t)q * d, sizeof(double) * d);
    s->removed[r] = 0; s->stuck[r] = 0; s->len[r] = 0;
    for (int j = 0; j < d; ++j) s->v[(size_t)r * d + j] = 0.0;
  }
  s->n_active = N - s->n_stuck;
  free(A); free(P); free(R); free(newx);
}

/* ------------------------------------------------------------------------------------------------
 * Phase 5: Hands Like Clouds.  The paper's Eq. 5 averages gradients at K perturbed
 * points; BASELINE.json north_star (e) fixes the zeroth-order form of the same smoothed gradient
 * (Eq. 9): ghat = (1/(M sigma)) sum_k f(x + sigma u_k) u_k, u_k ~ N(0, I) (R-11).
 * hlc_baseline = 1 subtracts the mean of the M values (control variate, same expectation).
 * ---------------------------------------------------------------------------------------------- */
/* The paper's own form, Eq. 5: theta <- theta + eta (1/K) sum_k grad f(theta + sigma z_k),
 * z_k ~ N(0, I), with finite-difference gradients: K 2d evaluations per step.  The draws z_k are
 * the same Philox normals as in the zeroth-order form; evaluation (k, +-h e_j) uses noise slot k 2d + 1 + 2j /
 * k 2d + 2 + 2j of (phase 5, step t).  Selected by hlc_baseline == 2 (DESIGN.md NEXT-2). */
static void hlc_sample_eq5(orc_ctx *s, int i, int t) {
  const int d = s->c.d, M = s->c.hlc_M;
  const double sig = s->sigma_eff, eta = (double)s->c.eta_hlc, h = (double)s->c.fd_h;
  double *gh = s->ghat + (size_t)i * d;
  for (int j = 0; j < d; ++j) gh[j] = 0.0;
  if (s->stuck[i] || s->removed[i]) return;            /* "Stuck samples are excluded" PAPER.md:120 */
  double *x = s->x + (size_t)i * d;
  double *pt = (double *)alloca(sizeof(double) * d), *xp = (double *)alloca(sizeof(double) * d);
  for (int k = 0; k < M; ++k) {
    for (int j = 0; j < d; ++j) {
      double u = orc_normal(s->c.seed, (uint32_t)i, (uint32_t)s->cycle, tag(5, t, PUR_HLC_U), (uint64_t)k * d + j);
      pt[j] = (double)(float)(x[j] + sig * u);          /* the perturbed point is an fp32 position like any other */
    }
    for (int j = 0; j < d; ++j) {
      memcpy(xp, pt, sizeof(double) * d);
      xp[j] = pt[j] + h;
      double fp = objective(s, xp) + orc_noise(s, s->cycle, i, 5, t, k * 2 * d + 1 + 2 * j);
      xp[j] = pt[j] - h;
      double fm = objective(s, xp) + orc_noise(s, s->cycle, i, 5, t, k * 2 * d + 2 + 2 * j);
      gh[j] += (fp - fm) / (2.0 * h) / M;
    }
  }
#pragma omp atomic
  s->evals[EV_HLC] += (uint64_t)M * 2 * d;
  for (int j = 0; j < d; ++j) x[j] = clipf32(x[j] + eta * gh[j], s->lo[j], s->hi[j]);
}

static void hlc_sample(orc_ctx *s, int i, int t) {
  const int d = s->c.d, M = s->c.hlc_M;
  const double sig = s->sigma_eff, eta = (double)s->c.eta_hlc;
  double *gh = s->ghat + (size_t)i * d;
  if (s->c.hlc_baseline == 2) { hlc_sample_eq5(s, i, t); return; }
  for (int j = 0; j < d; ++j) gh[j] = 0.0;
  if (s->stuck[i] || s->removed[i]) return;            /* "Stuck samples are excluded" PAPER.md:120 */
  double *x = s->x + (size_t)i * d;
  double *ubuf = s->hlc_u ? NULL : (double *)malloc(sizeof(double) * (size_t)M * d);
  double *u = s->hlc_u ? s->hlc_u + (size_t)i * M * d : ubuf, *fk = s->hlc_f + (size_t)i * M;
  double *pt = (double *)alloca(sizeof(double) * d);
  double fbar = 0.0;
  for (int k = 0; k < M; ++k) {
    for (int j = 0; j < d; ++j) {
      u[k * d + j] = orc_normal(s->c.seed, (uint32_t)i, (uint32_t)s->cycle, tag(5, t, PUR_HLC_U), (uint64_t)k * d + j);
      pt[j] = x[j] + sig * u[k * d + j];                /* evaluation points are not clipped (R-12) */
    }
    fk[k] = objective(s, pt) + orc_noise(s, s->cycle, i, 5, t, k);
    fbar += fk[k] / M;
  }
#pragma omp atomic
  s->evals[EV_HLC] += (uint64_t)M;
  double b = s->c.hlc_baseline ? fbar : 0.0;
  for (int j = 0; j < d; ++j) {
    double acc = 0.0;
    for (int k = 0; k < M; ++k) acc += (fk[k] - b) * u[k * d + j];
    gh[j] = acc / (M * sig);
  }
  for (int j = 0; j < d; ++j) x[j] = clipf32(x[j] + eta * gh[j], s->lo[j], s->hi[j]);
  free(ubuf);
}

/* Smoothing scale: supplied by the caller (sigma_s > 0), or auto-estimated from the sample spread,
 * sigma = c std({x_i : not stuck_i}) with c = |sigma_s| (paper default c = 0.1).  Reading R-18: std is the pooled
 * population standard deviation over all coordinates of the unfrozen samples, re-estimated at the start of every
 * Hands-Like-Clouds step; sigma = 0 (no spread, or nobody unfrozen) leaves the samples where they are. */
static void hlc_sigma(orc_ctx *s) {
  if (s->c.sigma_s > 0.0f) { s->sigma_eff = (double)s->c.sigma_s; return; }
  const int N = s->c.N, d = s->c.d;
  double n = 0.0, mean = 0.0, var = 0.0;
  for (int i = 0; i < N; ++i) if (!s->stuck[i] && !s->removed[i]) for (int j = 0; j < d; ++j) { mean += s->x[(size_t)i * d + j]; n += 1.0; }
  if (n == 0.0) { s->sigma_eff = 0.0; return; }
  mean /= n;
  for (int i = 0; i < N; ++i) if (!s->stuck[i] && !s->removed[i]) for (int j = 0; j < d; ++j) { double t = s->x[(size_t)i * d + j] - mean; var += t * t; }
  s->sigma_eff = fabs((double)s->c.sigma_s) * sqrt(var / n);
}

static void phase_hlc_step(orc_ctx *s, int t) {
  const int N = s->c.N;
  if (!(s->c.phase_mask & (1u << 5))) return;
  hlc_sigma(s);
  if (s->sigma_eff == 0.0) return;
#pragma omp parallel for schedule(dynamic, 8) num_threads(s->nthreads)
  for (int i = 0; i < N; ++i) hlc_sample(s, i, t);
}

/* ------------------------------------------------------------------------------------------------
 * Phase 6: momentum anti-convergence, Eq. 6: v <- mu v - alpha grad f, x <- x + v,
 * unfrozen samples only; v_0 = 0 at the start of the phase, x clipped to Theta (R-12).
 * ---------------------------------------------------------------------------------------------- */
static void anti_sample(orc_ctx *s, int i, int t) {
  const int d = s->c.d;
  const double mu = (double)s->c.mu, al = (double)s->c.alpha_anti;
  if (s->stuck[i] || s->removed[i]) return;            /* "Stuck samples are excluded" PAPER.md:129 */
  double *x = s->x + (size_t)i * d, *v = s->v + (size_t)i * d;
  double *gg = (double *)alloca(sizeof(double) * d), fdummy;
  if (t == 1) for (int j = 0; j < d; ++j) v[j] = 0.0;
  eval_fd(s, i, x, 6, t, 0, &fdummy, gg, EV_ANTI);
  for (int j = 0; j < d; ++j) {
    v[j] = (double)(float)(mu * v[j] - al * gg[j]);
    x[j] = clipf32(x[j] + v[j], s->lo[j], s->hi[j]);
  }
}

static void phase_anti_step(orc_ctx *s, int t) {
  const int N = s->c.N;
  if (!(s->c.phase_mask & (1u << 6))) return;
#pragma omp parallel for schedule(dynamic, 8) num_threads(s->nthreads)
  for (int i = 0; i < N; ++i) anti_sample(s, i, t);
}

/* ------------------------------------------------------------------------------------------------
 * Algorithm 1: one oscillation cycle.
 * ---------------------------------------------------------------------------------------------- */
int orc_phase(orc_ctx *s, int phase_id, int iter) {
  switch (phase_id) {
  case ORC_PH_RELEASE_EVAL: phase_release_eval(s); return 0;
  case ORC_PH_LBFGS_ITER:   phase_lbfgs_iter(s, iter); return 0;
  case ORC_PH_STICK:        phase_stick(s); return 0;
  case ORC_PH_DEDUP:        phase_dedup(s); return 0;
  case ORC_PH_RESEED:       phase_reseed(s); return 0;
  case ORC_PH_HLC_STEP:     phase_hlc_step(s, iter); return 0;
  case ORC_PH_ANTI_STEP:    phase_anti_step(s, iter); return 0;
  }
  return -1;
}

void orc_stats_now(orc_ctx *s, orc_stats *out) {
  out->cycle = s->cycle; out->n_stuck = s->n_stuck; out->k_lost = s->k_lost; out->n_active = s->n_active;
  out->reseed_strategy = s->reseed_strategy; out->gr_enabled = s->gr_enabled; out->f_max = s->f_max;
  memcpy(out->evals, s->evals, sizeof(s->evals));
}

int orc_step(orc_ctx *s, orc_stats *out) {
  if (s->cycle >= s->c.n_osc) return -5;
  s->cycle += 1;                                            /* "for k = 1..n_osc" */
  phase_release_eval(s);                                    /* Phase 1: release all, then converge */
  for (int it = 1; it <= s->c.n_conv; ++it) phase_lbfgs_iter(s, it);
  phase_stick(s);                                           /* Phase 2 */
  phase_dedup(s);                                           /* Phase 3 */
  s->reseed_strategy = 0;
  if (s->cycle < s->c.n_osc) {                              /* "if k < n_osc" */
    phase_reseed(s);                                        /* Phase 4 */
    for (int t = 1; t <= s->c.n_cloud; ++t) phase_hlc_step(s, t);   /* Phase 5 */
    for (int t = 1; t <= s->c.n_anti; ++t) phase_anti_step(s, t);   /* Phase 6 */
  }
  if (out) orc_stats_now(s, out);
  return 0;
}

/* "return {x_i : stuck_i}", sorted by (f descending, index ascending) */
typedef struct { double f; int idx; } mode_key;
static int mode_cmp(const void *a, const void *b) {
  const mode_key *p = (const mode_key *)a, *q = (const mode_key *)b;
  if (p->f > q->f) return -1;
  if (p->f < q->f) return 1;
  return (p->idx > q->idx) - (p->idx < q->idx);
}
int orc_modes(orc_ctx *s, double *modes, double *f, int32_t *idx, int32_t cap, int32_t *n_modes) {
  const int N = s->c.N, d = s->c.d;
  mode_key *k = (mode_key *)malloc(sizeof(mode_key) * N);
  int n = 0;
  for (int i = 0; i < N; ++i) if (s->stuck[i]) { k[n].f = s->f[i]; k[n].idx = i; ++n; }
  qsort(k, n, sizeof(mode_key), mode_cmp);
  *n_modes = n;
  int rc = (n > cap) ? -3 : 0;
  for (int q = 0; q < n && q < cap; ++q) {
    if (modes) memcpy(modes + (size_t)q * d, s->x + (size_t)k[q].idx * d, sizeof(double) * d);
    if (f) f[q] = k[q].f;
    if (idx) idx[q] = k[q].idx;
  }
  free(k);
  return rc;
}

/* ------------------------------------------------------------------------------------------------
 * Construction and state exchange.
 * ---------------------------------------------------------------------------------------------- */
static double *promote(const float *src, size_t n) {
  double *dst = (double *)malloc(sizeof(double) * (n ? n : 1));
  for (size_t i = 0; i < n; ++i) dst[i] = (double)src[i];
  return dst;
}
static double *dalloc(size_t n) { return (double *)calloc(n ? n : 1, sizeof(double)); }
#define DALLOC(n) dalloc((size_t)(n))

orc_ctx *orc_create(const orc_config *cfg, const orc_objective *obj, const float *x0) {
  if (!cfg || !obj || cfg->d != obj->d || cfg->d < 1 || cfg->N < 0 || cfg->lbfgs_m < 1 || cfg->lbfgs_m > 64)
    return NULL;
  orc_ctx *s = (orc_ctx *)calloc(1, sizeof(orc_ctx));
  s->c = *cfg; s->o = *obj; s->nthreads = 1;
  const size_t d = cfg->d, N = cfg->N, K = obj->K, m = cfg->lbfgs_m, M = cfg->hlc_M;
  s->lo = promote(cfg->lo, d); s->hi = promote(cfg->hi, d);
  size_t nmeans = 0, nmats = 0, na = 0, nb = 0;
  switch (obj->id) {
  case 0: nmeans = K * d; nmats = 1; na = K; break;
  case 1: nmeans = K * d; nmats = K * d; na = K; break;
  case 2: nmeans = K * d; nmats = K * d * d; na = K; break;
  case 3: nmats = K * d; na = K; nb = K; break;
  case 4: nmeans = d; nmats = d * d; break;
  case 5: case 6: case 7: case 8: case 9: case 10: break;       /* parameter-free (App. D) */
  case 11: if (d != 2) { free(s); return NULL; } break;
  default: free(s); return NULL;
  }
  s->means = promote(obj->means, nmeans); s->mats = promote(obj->mats, nmats);
  s->va = promote(obj->vec_a, na); s->vb = promote(obj->vec_b, nb);
  s->s0 = (double)obj->scalar0; s->sigma_noise = (double)obj->sigma_noise;
  s->x = promote(x0, N * d);
  s->f = DALLOC(N); s->g = DALLOC(N * d); s->v = DALLOC(N * d);
  s->S = DALLOC(N * m * d); s->Y = DALLOC(N * m * d);
  s->len = (int32_t *)calloc(N ? N : 1, sizeof(int32_t));
  s->stuck = (uint8_t *)calloc(N ? N : 1, 1); s->removed = (uint8_t *)calloc(N ? N : 1, 1);
  s->stalled = (uint8_t *)calloc(N ? N : 1, 1);
  s->p = DALLOC(N * d); s->ls_margin = DALLOC(N); s->asc_margin = DALLOC(N); s->curv_margin = DALLOC(N);
  s->ghat = DALLOC(N * d); s->hlc_f = DALLOC(N * M); s->hlc_u = (N * M * d <= ((size_t)1 << 25)) ? DALLOC(N * M * d) : NULL; s->rs_margin = DALLOC(N);
  s->ls_b = (int32_t *)calloc(N ? N : 1, sizeof(int32_t));
  s->rs_src = (int32_t *)calloc(N ? N : 1, sizeof(int32_t));
  s->rs_cand = (int32_t *)calloc(N ? N : 1, sizeof(int32_t));
  s->rs_score = DALLOC(N * 16);
  s->gr_enabled = 1; s->f_max = -INFINITY;
  return s;
}

void orc_destroy(orc_ctx *s) {
  if (!s) return;
  free(s->lo); free(s->hi); free(s->means); free(s->mats); free(s->va); free(s->vb);
  free(s->x); free(s->f); free(s->g); free(s->v); free(s->S); free(s->Y); free(s->len);
  free(s->stuck); free(s->removed); free(s->stalled); free(s->p); free(s->ls_margin); free(s->asc_margin);
  free(s->curv_margin); free(s->ghat); free(s->hlc_f); free(s->hlc_u); free(s->rs_margin);
  free(s->ls_b); free(s->rs_src); free(s->rs_cand); free(s->rs_score);
  free(s);
}

void orc_set_threads(orc_ctx *s, int n) { s->nthreads = n > 0 ? n : 1; }

static int xfer(void *state, size_t bytes_state, void *user, uint64_t bytes_user, int to_user) {
  if (bytes_user != bytes_state) return -1;
  if (to_user) memcpy(user, state, bytes_state); else memcpy(state, user, bytes_state);
  return 0;
}

/* history is kept [N][m][d]; it is exchanged as [m][N][d] (slot 0 = oldest) */
static int xfer_hist(orc_ctx *s, double *H, double *user, uint64_t bytes, int to_user) {
  const size_t d = s->c.d, N = s->c.N, m = s->c.lbfgs_m;
  if (bytes != sizeof(double) * N * m * d) return -1;
  for (size_t i = 0; i < N; ++i)
    for (size_t l = 0; l < m; ++l)
      for (size_t j = 0; j < d; ++j) {
        double *a = H + (i * m + l) * d + j, *b = user + (l * N + i) * d + j;
        if (to_user) *b = *a; else *a = *b;
      }
  return 0;
}

static int xfer_field(orc_ctx *s, int field, void *u, uint64_t bytes, int to_user) {
  const size_t d = s->c.d, N = s->c.N, M = s->c.hlc_M;
  switch (field) {
  case ORC_X: return xfer(s->x, 8 * N * d, u, bytes, to_user);
  case ORC_F: return xfer(s->f, 8 * N, u, bytes, to_user);
  case ORC_G: return xfer(s->g, 8 * N * d, u, bytes, to_user);
  case ORC_V: return xfer(s->v, 8 * N * d, u, bytes, to_user);
  case ORC_STUCK: return xfer(s->stuck, N, u, bytes, to_user);
  case ORC_REMOVED: return xfer(s->removed, N, u, bytes, to_user);
  case ORC_STALLED: return xfer(s->stalled, N, u, bytes, to_user);
  case ORC_HIST_S: return xfer_hist(s, s->S, (double *)u, bytes, to_user);
  case ORC_HIST_Y: return xfer_hist(s, s->Y, (double *)u, bytes, to_user);
  case ORC_HIST_LEN: return xfer(s->len, 4 * N, u, bytes, to_user);
  case ORC_CTRL: {
    int32_t c[8] = { s->cycle, s->gr_enabled, s->gr_unproductive, s->gr_prev_modes, s->gr_used_last,
                     s->k_lost, s->n_stuck, s->n_active };
    if (bytes != sizeof(c)) return -1;
    if (to_user) memcpy(u, c, sizeof(c));
    else {
      memcpy(c, u, sizeof(c));
      s->cycle = c[0]; s->gr_enabled = c[1]; s->gr_unproductive = c[2]; s->gr_prev_modes = c[3];
      s->gr_used_last = c[4]; s->k_lost = c[5]; s->n_stuck = c[6]; s->n_active = c[7];
    }
    return 0;
  }
  case ORC_P: return xfer(s->p, 8 * N * d, u, bytes, to_user);
  case ORC_LS_B: return xfer(s->ls_b, 4 * N, u, bytes, to_user);
  case ORC_LS_MARGIN: return xfer(s->ls_margin, 8 * N, u, bytes, to_user);
  case ORC_ASC_MARGIN: return xfer(s->asc_margin, 8 * N, u, bytes, to_user);
  case ORC_CURV_MARGIN: return xfer(s->curv_margin, 8 * N, u, bytes, to_user);
  case ORC_GHAT: return xfer(s->ghat, 8 * N * d, u, bytes, to_user);
  case ORC_HLC_F: return xfer(s->hlc_f, 8 * N * M, u, bytes, to_user);
  case ORC_HLC_U: return s->hlc_u ? xfer(s->hlc_u, 8 * N * M * d, u, bytes, to_user) : -1;
  case ORC_RS_SRC: return xfer(s->rs_src, 4 * N, u, bytes, to_user);
  case ORC_RS_CAND: return xfer(s->rs_cand, 4 * N, u, bytes, to_user);
  case ORC_RS_MARGIN: return xfer(s->rs_margin, 8 * N, u, bytes, to_user);
  case ORC_RS_SCORE: return xfer(s->rs_score, 8 * N * 16, u, bytes, to_user);
  case ORC_SIGMA: return to_user ? xfer(&s->sigma_eff, 8, u, bytes, 1) : -1;
  }
  return -1;
}
int orc_get(orc_ctx *s, int field, void *dst, uint64_t bytes) { return xfer_field(s, field, dst, bytes, 1); }
int orc_set(orc_ctx *s, int field, const void *src, uint64_t bytes) { return xfer_field(s, field, (void *)src, bytes, 0); }
