// chisao_common.cuh -- shared definitions of the CUDA path (host + device).  sm_100a only.
//
// Nothing here is shared with oracle/: the Philox generator, the objective arithmetic and every phase
// are restated independently on this side.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/chisao.h"

namespace chisao {

// ---- evaluation tiling -------------------------------------------------------------------------
constexpr int NT = 128;          // threads per evaluation CTA
constexpr int PPT = 2;           // points evaluated per thread (register tile)
constexpr int PTILE = NT * PPT;  // points per CTA tile
constexpr int CHUNK_BYTES = 20 * 1024;  // objective-parameter chunk staged in SMEM per buffer

// ---- Philox purposes / evaluation counters (R-15, R-2) -----------------------------------------
enum { PUR_INIT = 0, PUR_NOISE = 1, PUR_HLC_U = 2, PUR_RS_SRC = 3, PUR_RS_T = 4, PUR_RS_DIR = 5,
       PUR_GR_MATRIX = 6, PUR_RS_UNIF = 7 };
enum { EV_INIT = 0, EV_LS = 1, EV_LBFGS_FD = 2, EV_HLC = 5, EV_ANTI = 6 };

// ---- device control block (one per context, lives in the workspace) ----------------------------
// populations up to this size run an ordered scan as ONE launch (k_scan_small), larger ones as three (chisao_select.cu)
constexpr int SCAN_SMALL_MAX = 4096;
__host__ __device__ inline int scan_launches(int N) { return (N == 0 || N <= SCAN_SMALL_MAX) ? 1 : 3; }

struct Ctrl {
  int32_t cycle, gr_enabled, gr_unproductive, gr_prev_modes, gr_used_last, k_lost, n_stuck, n_active;
  int32_t strategy;        // reseed strategy of the current cycle
  int32_t nA, nP, nR;      // list lengths after dedup (ascending lists A, P, R)
  int32_t nP0;             // stuck count before dedup
  int32_t nE;              // explore-list length (not stuck, not removed) for phases 5-6
  uint32_t fmax_enc;       // order-preserving image of f_max (0 = nothing finite yet)
  int32_t ls_cnt[3];       // rotating line-search worklist counters
  int32_t fd_cnt;          // samples whose trial was accepted this iteration
  float sigma_eff;         // smoothing scale used by the current HLC step (caller's, or c * std of the unfrozen samples)
  unsigned long long evals[8];
  double sx, sxx;          // pooled sums for the sigma auto-estimate
};

// ---- objective parameters packed as fixed-size component records --------------------------------
// record r of an objective = `rec` floats (multiple of 4), coordinates padded to DP with zeros:
//   GMM_ISO : mu[DP] | a, 0, 0, 0                       s0 = 1/(2 sigma^2)
//   GMM_DIAG: mu[DP] | inv[DP] | a, 0, 0, 0
//   GMM_FULL: W[DP][DP] | mu[DP] | a, 0, 0, 0
//   RFF     : w[DP] as fp64 (2 DP floats) | a, b, 0, 0    s0 = quadratic coefficient
//   QUAD    : W[DP][DP] | c[DP] | 0, 0, 0, 0
//   ids >= 5 (Appendix D): no parameters; the evaluator is instantiated once (template OBJ = CHISAO_OBJ_APPD) and
//             picks the function from DevObj::id
constexpr int CHISAO_OBJ_APPD = 5;
struct DevObj {
  int32_t id, d, K, DP;
  int32_t rec;             // floats per record
  int32_t kc;              // records per SMEM chunk
  float s0, sigma_noise;
  const float *recs;       // device, [K][rec], 16-byte aligned
};

inline int padded_dim(int d) { return d <= 8 ? 8 : (d <= 32 ? 32 : 64); }
inline size_t history_plane_floats(size_t N, size_t d) { return N * d + 2112; }   // + 8448 bytes = 33 x 256: rows stay 256-byte aligned at d = 64
inline int record_floats(int id, int DP) {
  switch (id) {
    case CHISAO_OBJ_GMM_ISO: return DP + 4;
    case CHISAO_OBJ_GMM_DIAG: return 2 * DP + 4;
    case CHISAO_OBJ_GMM_FULL: return DP * DP + DP + 4;
    case CHISAO_OBJ_RFF: return 2 * DP + 4;
    case CHISAO_OBJ_QUAD: return DP * DP + DP + 4;
  }
  return 4;   // Appendix-D functions carry no parameters (one dummy record keeps the workspace carve uniform)
}

// ---- device state pointers ------------------------------------------------------------------------
struct State {
  int32_t N, d, m, M;
  float *x, *f, *g, *v, *xt, *ft, *gn, *p, *dec, *tcur, *ginf;
  float *S, *Y;                       // [m] planes of [N][d] (physical ring slots), `hplane` floats apart
  size_t hplane;                      // plane stride in floats: N d plus a pad that keeps the planes of one sample from
                                      // sitting a power of two apart (at C5 N d 4 = 2^24 bytes: every one of a sample's 2 m
                                      // history rows would map to the same DRAM channel / bank group)
  int32_t *hist_len, *hist_head, *ls_b;
  uint8_t *stuck, *removed, *stalled;
  int32_t *listA, *listP, *listR, *listE, *listP0, *ls_list[3], *fd_list;
  int32_t *blk_cnt;                   // scan scratch [3][nb] counts then offsets
  float *ghat, *hlc_f, *grQ, *lo, *hi;
  int32_t *rs_src, *rs_cand;
  Ctrl *ctrl;
};

struct Hyper {                        // by-value copy of the cycle hyper-parameters
  int32_t n_osc, n_conv, n_anti, n_cloud, hlc_M, lbfgs_m, ls_max, reseed_cands, hlc_baseline;
  uint32_t phase_mask;
  float fd_h, eps_grad, eps_dup, log_delta, mu, alpha_anti, eta_hlc, sigma_s, ls_c1, ls_shrink;
  uint64_t seed;
};

// modes of the evaluation kernels
enum { FD_GRAD = 0, FD_ANTI = 1 };
enum { PT_CENTRE = 0, PT_LS = 1, PT_LS_ALL = 2 };
// modes of the list-building scan
enum { SCAN_STICK = 0, SCAN_FINAL = 1, SCAN_EXPLORE = 2, SCAN_STICK_FLAGS = 3 };

// launchers implemented in the .cu files (all enqueue on `st`, return the cudaError of the launch)
cudaError_t launch_eval_fd(const DevObj &o, const State &s, const Hyper &h, int cycle, const float *X,
                           const int32_t *list, const int32_t *count, int max_count, int mode, float *g_out,
                           int phase, int iter, int counter, cudaStream_t st);
cudaError_t launch_eval_points(const DevObj &o, const State &s, const Hyper &h, int cycle, int mode, int b,
                               int iter, cudaStream_t st);
cudaError_t launch_hlc(const DevObj &o, const State &s, const Hyper &h, int cycle, int iter, cudaStream_t st);
cudaError_t eval_kernels_configure();   // opt-in dynamic shared memory for every instantiation

// mode: 0 direction only (stand-alone unit), 1 first iteration of a cycle (release folded in), 2 update of the previous
// iteration + direction (chisao_lbfgs.cu)
cudaError_t launch_lbfgs_step(const State &s, const Hyper &h, int mode, int it, cudaStream_t st);
cudaError_t launch_lbfgs_update(const State &s, const Hyper &h, bool stick_partials, cudaStream_t st);
cudaError_t launch_release(const State &s, cudaStream_t st);
cudaError_t launch_stick(const State &s, const Hyper &h, bool have_partials, cudaStream_t st);   // ginf, f_max, flags, P0
cudaError_t launch_dedup(const State &s, const Hyper &h, bool rebuild_p0, cudaStream_t st);   // removed + lists + GR state
cudaError_t launch_reseed(const State &s, const Hyper &h, int cycle, bool standalone, cudaStream_t st);
cudaError_t launch_explore_list(const State &s, cudaStream_t st);
// paper-form HLC (Eq. 5) helpers: stage 0 perturb (xt = x + sigma z_k), 1 accumulate (ghat += gn / M), 2 apply
cudaError_t launch_hlc_sigma(const State &s, const Hyper &h, cudaStream_t st);   // ctrl->sigma_eff (R-18)
cudaError_t launch_hlc5(const State &s, const Hyper &h, int cycle, int iter, int k, int stage, cudaStream_t st);
cudaError_t launch_seed_population(const State &s, const Hyper &h, cudaStream_t st);
cudaError_t launch_gather_rows(const float *x, const int32_t *idx, int n, int d, float *out, cudaStream_t st);

}  // namespace chisao
