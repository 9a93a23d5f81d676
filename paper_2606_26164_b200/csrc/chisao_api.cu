// chisao_api.cu -- host side of the C ABI declared in include/chisao.h: validation, workspace carving,
// parameter packing, the per-cycle launch sequence (Algorithm 1) and state exchange.
// Every step of the path runs in the kernels; the host only enqueues.  There is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "chisao_eval_kernels.cuh"
#include "chisao_resident.cuh"
#include <cuda_fp16.h>
#include "chisao_tc.cuh"

using namespace chisao;

namespace {

thread_local std::string g_last_error;

struct Segment { size_t off, bytes; };

struct Layout {
  size_t total = 0;
  size_t take(size_t bytes) {
    const size_t off = total;
    total += (bytes + 255) & ~size_t(255);
    return off;
  }
};

struct TimedRec { int cls; cudaEvent_t a, b; };

}  // namespace

// for the entry points that live in other translation units (chisao_static.cu): the text chisao_last_error(NULL) returns
namespace chisao { void set_global_error(const char *msg) { g_last_error = msg ? msg : ""; } }

struct chisao_ctx {
  chisao_config cfg;
  Hyper hp;
  DevObj obj;
  State st;
  cudaStream_t stream;
  int cycle = 0;
  std::vector<float> lo, hi, recs_host, tc_host;
  TcObj tc;
  bool use_tc = false;   // dense objective at d > 32: tensor-core evaluator (chisao_tc.cuh)
  bool stencil_aware = false;   // chisao_set_option(CHISAO_OPT_STENCIL_AWARE): FD gradients by chisao_stencil.cu
  std::string err;
  uint64_t launches = 0;
  uint32_t timing = 0;   // bit k: kernel class k is bracketed with CUDA events
  std::vector<TimedRec> recs;
  std::vector<cudaEvent_t> pool;
  size_t ws_bytes = 0;
  // one cycle as a CUDA graph (chisao_step): captured on an internal stream that is forked from / joined to the
  // caller's stream with events, re-captured every cycle (the cycle index is a kernel argument) and applied to the
  // instantiated graph with cudaGraphExecUpdate; slot 0 = full cycle, 1 = the short last cycle
  bool graph_on = true;
  cudaStream_t gstream = nullptr;
  cudaEvent_t gfork = nullptr, gjoin = nullptr;
  cudaGraphExec_t gexec[2] = {nullptr, nullptr};
  uint64_t graph_launches = 0;
  // line search: every trial of a tile in one launch (PT_LS_ALL) when a tile of the evaluator costs microseconds
  // (FP32-FMA evaluators of the small objectives, QUAD and RFF on the tensor cores); one launch per trial on compacted
  // worklists otherwise (GMM_FULL: a tile streams the whole mixture, the retries must stay dense)
  bool ls_tile_local = false;
  // Phase 1 as ONE launch with the (s, y) history in registers (chisao_resident.cuh): FP32-FMA evaluators, d a power of
  // two <= 32, parameters in one chunk, m <= 16
  bool resident = false, resident_ok = false;
  bool in_cycle = false; // enqueue_cycle is running: the launch sequence may rely on what the previous unit left behind
};

namespace {

int fail(chisao_ctx *c, int code, const std::string &msg) {
  g_last_error = msg;
  if (c) c->err = msg;
  return code;
}
int cuda_fail(chisao_ctx *c, cudaError_t e, const char *what) {
  return fail(c, CHISAO_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                                   \
  do {                                                             \
    cudaError_t e_ = (call);                                       \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);       \
  } while (0)

int validate(const chisao_config *cfg, const chisao_objective *obj, std::string &why) {
  if (!cfg || !obj) { why = "null config/objective"; return CHISAO_E_INVALID; }
  if (cfg->d < 1 || cfg->d > CHISAO_MAX_D) { why = "d must be in 1..64"; return CHISAO_E_INVALID; }
  if (obj->d != cfg->d) { why = "objective.d != config.d"; return CHISAO_E_INVALID; }
  if (cfg->N < 0) { why = "N < 0"; return CHISAO_E_INVALID; }
  if (cfg->lbfgs_m < 1 || cfg->lbfgs_m > CHISAO_MAX_M) { why = "lbfgs_m must be in 1..16"; return CHISAO_E_INVALID; }
  if (cfg->hlc_M < 1 || cfg->hlc_M > PTILE) { why = "hlc_M must be in 1..256"; return CHISAO_E_INVALID; }
  if (cfg->ls_max < 0 || cfg->ls_max > 30) { why = "ls_max must be in 0..30"; return CHISAO_E_INVALID; }
  if (cfg->reseed_cands < 1 || cfg->reseed_cands > 16) { why = "reseed_cands must be in 1..16"; return CHISAO_E_INVALID; }
  if (cfg->n_osc < 1 || cfg->n_conv < 0 || cfg->n_anti < 0 || cfg->n_cloud < 0) { why = "negative iteration count"; return CHISAO_E_INVALID; }
  if (!(cfg->fd_h > 0.0f)) { why = "fd_h must be > 0"; return CHISAO_E_INVALID; }
  if (!(cfg->sigma_s != 0.0f) || !(fabsf(cfg->sigma_s) < 3.0e38f)) { why = "sigma_s must be > 0 (given) or < 0 (auto, c = |sigma_s|)"; return CHISAO_E_INVALID; }
  if (!cfg->lo || !cfg->hi) { why = "null bounds"; return CHISAO_E_INVALID; }
  for (int j = 0; j < cfg->d; ++j)
    if (!(cfg->lo[j] <= cfg->hi[j])) { why = "lo > hi"; return CHISAO_E_INVALID; }
  if (obj->id < 0 || obj->id > CHISAO_OBJ_BUKIN6) { why = "unknown objective id"; return CHISAO_E_INVALID; }
  if (obj->K < 1) { why = "K < 1"; return CHISAO_E_INVALID; }
  if (obj->id >= CHISAO_OBJ_RASTRIGIN) {
    if (obj->K != 1) { why = "Appendix-D objectives need K = 1"; return CHISAO_E_INVALID; }
    if (obj->id == CHISAO_OBJ_BUKIN6 && obj->d != 2) { why = "Bukin N.6 needs d = 2"; return CHISAO_E_INVALID; }
  } else {
    if (obj->id == CHISAO_OBJ_QUAD && obj->K != 1) { why = "QUAD needs K = 1"; return CHISAO_E_INVALID; }
    if (!obj->mats) { why = "objective.mats is null"; return CHISAO_E_INVALID; }
    if (obj->id != CHISAO_OBJ_RFF && !obj->means) { why = "objective.means is null"; return CHISAO_E_INVALID; }
    if (obj->id != CHISAO_OBJ_QUAD && !obj->vec_a) { why = "objective.vec_a is null"; return CHISAO_E_INVALID; }
    if (obj->id == CHISAO_OBJ_RFF && !obj->vec_b) { why = "objective.vec_b is null"; return CHISAO_E_INVALID; }
  }
  if (!(obj->sigma_noise >= 0.0f)) { why = "sigma_noise < 0"; return CHISAO_E_INVALID; }
  return CHISAO_OK;
}

// workspace carve; fills st pointers relative to `base` (may be null when only sizing)
// RFF on the tensor cores (chisao_tc.cuh, tc_rff_tile): d <= 32, K <= 256 and value ranges inside the fixed-point
// split: |x| < 2^ex (box radius + HLC spread + FD step), |w| < 2^ew, with ex, ew in [-6, 10]
// largest |coordinate| an evaluation point can have: box radius + the Hands-Like-Clouds spread (8 sigma; with the auto
// estimate sigma_s < 0, sigma = |sigma_s| x pooled std of the unfrozen samples <= |sigma_s| x box diameter) + the FD step
float eval_point_radius(const chisao_config &c) {
  float rad = 0.f;
  for (int j = 0; j < c.d; ++j) rad = std::max(rad, std::max(std::fabs(c.lo[j]), std::fabs(c.hi[j])));
  const float sig = c.sigma_s > 0.0f ? c.sigma_s : 2.0f * rad * std::fabs(c.sigma_s);
  return rad + 8.0f * sig + std::fabs(c.fd_h);
}
bool rff_tc_scales(const chisao_objective &o, const chisao_config &c, int *ex_out, int *ew_out) {
  if (o.id != CHISAO_OBJ_RFF || o.d > RFF_TC_D || o.K > RFF_TC_K || getenv("CHISAO_RFF_FP64")) return false;
  float wmax = 0.f;
  for (size_t e = 0; e < (size_t)o.K * o.d; ++e) wmax = std::max(wmax, std::fabs(o.mats[e]));
  const float xmax = eval_point_radius(c);
  if (!(wmax > 0.f) || !(xmax > 0.f) || !(wmax < 3.0e38f) || !(xmax < 3.0e38f)) return false;
  int ex = 0, ew = 0;
  std::frexp(xmax, &ex);   // xmax = m 2^ex, m in [0.5, 1): xmax < 2^ex (or = 2^(ex-1): still inside the 4x headroom)
  std::frexp(wmax, &ew);
  ew += 0;
  if (ex < -6 || ex > 10 || ew < -6 || ew > 10 || ex + ew > 14) return false;   // uA = 2^(ex+ew-18) <= 1/16: 2 pi / uA > 100
  if (ex_out) *ex_out = ex;
  if (ew_out) *ew_out = ew;
  return true;
}
inline bool wants_tc(const chisao_objective &o, const chisao_config &c) {
  return ((o.id == CHISAO_OBJ_GMM_FULL || o.id == CHISAO_OBJ_QUAD) && o.d > 32) || rff_tc_scales(o, c, nullptr, nullptr);
}

size_t carve(const chisao_config &c, const chisao_objective &o, unsigned char *base, State *st, const float **recs_dev,
             const float **tc_dev = nullptr) {
  Layout L;
  const size_t N = (size_t)c.N, d = (size_t)c.d, m = (size_t)c.lbfgs_m, M = (size_t)c.hlc_M;
  const int DP = padded_dim(c.d);
  const size_t rec = (size_t)record_floats(o.id, DP);
  const size_t nb = (N + 1023) / 1024;
  auto F = [&](size_t n) { return L.take(n * 4); };
  const size_t o_ctrl = L.take(sizeof(Ctrl));
  const size_t o_recs = F((size_t)o.K * rec);
  const size_t o_lo = F(d), o_hi = F(d);
  const size_t o_f = F(N), o_ft = F(N), o_dec = F(N), o_tcur = F(N), o_ginf = F(N);
  const size_t o_g = F(N * d), o_v = F(N * d), o_xt = F(N * d), o_gn = F(N * d), o_p = F(N * d), o_gh = F(N * d);
  const size_t hp_ = history_plane_floats(N, d);
  const size_t o_S = F(m * hp_), o_Y = F(m * hp_);
  const size_t o_hl = F(N), o_hh = F(N), o_lsb = F(N), o_rss = F(N), o_rsc = F(N);
  const size_t o_st = L.take(N), o_rm = L.take(N), o_sl = L.take(N);
  size_t o_lists[9];
  for (auto &x : o_lists) x = F(N);
  const size_t o_blk = F(3 * nb + 3);
  const size_t o_hf = F(N * M);
  const size_t o_q = F(d * d);
  const size_t o_tc = F(!wants_tc(o, c) ? 0 : (o.id == CHISAO_OBJ_RFF ? (size_t)RFF_REC_FLOATS : (o.id == CHISAO_OBJ_GMM_FULL ? (size_t)((o.K + 1) / 2) * TCX_REC : (size_t)o.K * TC_REC)));
  if (base && st) {
    auto P = [&](size_t off) { return reinterpret_cast<float *>(base + off); };
    auto I = [&](size_t off) { return reinterpret_cast<int32_t *>(base + off); };
    st->ctrl = reinterpret_cast<Ctrl *>(base + o_ctrl);
    *recs_dev = P(o_recs);
    st->lo = P(o_lo); st->hi = P(o_hi);
    st->f = P(o_f); st->ft = P(o_ft); st->dec = P(o_dec); st->tcur = P(o_tcur); st->ginf = P(o_ginf);
    st->g = P(o_g); st->v = P(o_v); st->xt = P(o_xt); st->gn = P(o_gn); st->p = P(o_p); st->ghat = P(o_gh);
    st->S = P(o_S); st->Y = P(o_Y); st->hplane = hp_;
    st->hist_len = I(o_hl); st->hist_head = I(o_hh); st->ls_b = I(o_lsb); st->rs_src = I(o_rss); st->rs_cand = I(o_rsc);
    st->stuck = base + o_st; st->removed = base + o_rm; st->stalled = base + o_sl;
    st->listA = I(o_lists[0]); st->listP = I(o_lists[1]); st->listR = I(o_lists[2]); st->listE = I(o_lists[3]);
    st->listP0 = I(o_lists[4]); st->ls_list[0] = I(o_lists[5]); st->ls_list[1] = I(o_lists[6]);
    st->ls_list[2] = I(o_lists[7]); st->fd_list = I(o_lists[8]);
    st->blk_cnt = I(o_blk);
    st->hlc_f = P(o_hf);
    st->grQ = P(o_q);
    if (tc_dev) *tc_dev = P(o_tc);
  }
  return L.total;
}

// pack the objective into fixed-size records (pure data movement; layouts in chisao_common.cuh)
void pack_records(const chisao_objective &o, int DP, std::vector<float> &out, float &s0) {
  const int d = o.d, K = o.K, rec = record_floats(o.id, DP);
  out.assign((size_t)K * rec, 0.0f);
  s0 = 0.0f;
  for (int k = 0; k < K; ++k) {
    float *r = out.data() + (size_t)k * rec;
    switch (o.id) {
      case CHISAO_OBJ_GMM_ISO:
        for (int j = 0; j < d; ++j) r[j] = o.means[(size_t)k * d + j];
        r[DP] = o.vec_a[k];
        break;
      case CHISAO_OBJ_GMM_DIAG:
        for (int j = 0; j < d; ++j) { r[j] = o.means[(size_t)k * d + j]; r[DP + j] = o.mats[(size_t)k * d + j]; }
        r[2 * DP] = o.vec_a[k];
        break;
      case CHISAO_OBJ_GMM_FULL:
      case CHISAO_OBJ_QUAD:
        for (int a = 0; a < d; ++a)
          for (int b = 0; b < d; ++b) r[a * DP + b] = o.mats[((size_t)k * d + a) * d + b];
        for (int j = 0; j < d; ++j) r[DP * DP + j] = o.means[(size_t)k * d + j];
        r[DP * DP + DP] = (o.id == CHISAO_OBJ_GMM_FULL) ? o.vec_a[k] : 0.0f;
        break;
      case CHISAO_OBJ_RFF:
        for (int j = 0; j < d; ++j) {   // exact promotion of the fp32 frequencies to fp64
          const double w = (double)o.mats[(size_t)k * d + j];
          std::memcpy(r + 2 * j, &w, sizeof(double));
        }
        r[2 * DP] = o.vec_a[k]; r[2 * DP + 1] = o.vec_b[k];
        break;
    }
  }
  if (o.id == CHISAO_OBJ_GMM_ISO) s0 = (float)(1.0 / (2.0 * (double)o.mats[0] * (double)o.mats[0]));
  if (o.id == CHISAO_OBJ_RFF) s0 = o.scalar0;
}

// tensor-core operand records: W_k split into tf32 hi / lo (round-to-nearest, ties away: the integer form of
// cvt.rna.tf32.f32) and stored in the canonical K-major UMMA layout, then mu_k and a_k (chisao_tc.cuh)
float tf32_rna_host(float x) {
  uint32_t u;
  std::memcpy(&u, &x, 4);
  if ((u & 0x7F800000u) != 0x7F800000u) u += 0x1000u;
  u &= 0xFFFFE000u;
  float r;
  std::memcpy(&r, &u, 4);
  return r;
}
void pack_tc_records(const chisao_objective &o, std::vector<float> &out) {
  const int d = o.d, K = o.K;
  out.assign((size_t)K * TC_REC, 0.0f);
  for (int k = 0; k < K; ++k) {
    float *r = out.data() + (size_t)k * TC_REC;
    for (int n = 0; n < d; ++n)
      for (int c = 0; c < d; ++c) {
        const float w = o.mats[((size_t)k * d + n) * d + c];
        const float h = tf32_rna_host(w), l = tf32_rna_host(w - h);
        const int idx = (c / 4) * 256 + n * 4 + (c % 4);
        r[idx] = h; r[TC_D * TC_D + idx] = l;
      }
    for (int j = 0; j < d; ++j) r[2 * TC_D * TC_D + j] = o.means[(size_t)k * d + j];
    r[2 * TC_D * TC_D + TC_D] = (o.id == CHISAO_OBJ_GMM_FULL) ? o.vec_a[k] : 0.0f;
  }
}

// QUAD record for kind::f16 (chisao_tc.cuh, tc_quad_run16): fp16 hi / lo images of 2^ws W -- element (n, c) at 16-bit index
// (c/8)*512 + n*8 + (c%8), hi image at byte 0, lo image at byte 8192 -- then c where the tf32 record has it
void pack_quad16_record(const chisao_objective &o, int ws, std::vector<float> &out) {
  const int d = o.d;
  out.assign((size_t)TC_REC, 0.0f);
  uint16_t *img = reinterpret_cast<uint16_t *>(out.data());
  for (int n = 0; n < d; ++n)
    for (int c = 0; c < d; ++c) {
      const float w = std::ldexp(o.mats[(size_t)n * d + c], ws);
      const __half h = __float2half_rn(w), l = __float2half_rn(w - __half2float(h));
      const size_t idx = (size_t)(c / 8) * 512 + (size_t)n * 8 + (c % 8);
      img[idx] = __half_as_ushort(h); img[4096 + idx] = __half_as_ushort(l);
    }
  for (int j = 0; j < d; ++j) out[2 * TC_D * TC_D + j] = o.means[j];
}
// scale of the QUAD fp16 images: max |2^ws W| in [4096, 8192); false if W is zero or not finite, or the tf32 form is forced
bool quad16_scale(const chisao_objective &o, int *ws) {
  float wmax = 0.f;
  for (size_t e = 0; e < (size_t)o.d * o.d; ++e) wmax = std::max(wmax, std::fabs(o.mats[e]));
  if (!(wmax > 0.f) || !std::isfinite(wmax) || getenv("CHISAO_TC_TF32")) return false;
  int e2 = 0;
  std::frexp(wmax, &e2);                      // wmax = m 2^e2, m in [0.5, 1)
  *ws = 13 - e2;                              // 2^ws wmax in [4096, 8192)
  return *ws >= -40 && *ws <= 40;
}

// x-stationary pair records of GMM_FULL (chisao_tc.cuh): B image of the pair [W_2p ; W_2p+1] (128 rows, hi then lo),
// c = W mu (fp64 product, rounded once), a; an odd K is padded with a zero component of weight a = -inf
void pack_tcx_records(const chisao_objective &o, std::vector<float> &out) {
  const int d = o.d, K = o.K, npair = (K + 1) / 2;
  out.assign((size_t)npair * TCX_REC, 0.0f);
  for (int p = 0; p < npair; ++p) {
    float *r = out.data() + (size_t)p * TCX_REC;
    for (int hf = 0; hf < 2; ++hf) {
      const int k = 2 * p + hf;
      if (k >= K) { r[TCX_W_FLOATS + 128 + hf] = -INFINITY; continue; }
      for (int n = 0; n < d; ++n) {
        double cn = 0.0;
        for (int c = 0; c < d; ++c) {
          const float w = o.mats[((size_t)k * d + n) * d + c];
          const float h = tf32_rna_host(w), l = tf32_rna_host(w - h);
          const int idx = (c / 4) * 512 + (64 * hf + n) * 4 + (c % 4);
          r[idx] = h; r[TCX_W_FLOATS / 2 + idx] = l;
          cn += (double)w * (double)o.means[(size_t)k * d + c];
        }
        r[TCX_W_FLOATS + 64 * hf + n] = (float)cn;
      }
      r[TCX_W_FLOATS + 128 + hf] = o.vec_a[k];
    }
  }
}

// the same pair records with fp16 hi / lo images (kind::f16): element (n, c) of an image at byte (c/8)*2048 + n*16 +
// (c%8)*2, hi image then lo image (16 KB each) at the start of the record; c and a as above
void pack_tcx16_records(const chisao_objective &o, std::vector<float> &out) {
  const int d = o.d, K = o.K, npair = (K + 1) / 2;
  out.assign((size_t)npair * TCX_REC, 0.0f);
  for (int p = 0; p < npair; ++p) {
    float *r = out.data() + (size_t)p * TCX_REC;
    uint16_t *img = reinterpret_cast<uint16_t *>(r);
    for (int hf = 0; hf < 2; ++hf) {
      const int k = 2 * p + hf;
      if (k >= K) { r[TCX_W_FLOATS + 128 + hf] = -INFINITY; continue; }
      for (int n = 0; n < d; ++n) {
        double cn = 0.0;
        for (int c = 0; c < d; ++c) {
          const float w = o.mats[((size_t)k * d + n) * d + c];
          const __half h = __float2half_rn(w), l = __float2half_rn(w - __half2float(h));
          const size_t idx = (size_t)(c / 8) * 1024 + (size_t)(64 * hf + n) * 8 + (c % 8);   // in 16-bit elements
          img[idx] = __half_as_ushort(h); img[8192 + idx] = __half_as_ushort(l);
          cn += (double)w * (double)o.means[(size_t)k * d + c];
        }
        r[TCX_W_FLOATS + 64 * hf + n] = (float)cn;
        // -c_n as three fp16 pieces (33 bits) in K positions 0..2 of the extra K = 16 step, 32 KB into the record
        const __half c1 = __float2half_rn((float)-cn);
        const double r1 = -cn - (double)__half2float(c1);
        const __half c2 = __float2half_rn((float)r1);
        const __half c3 = __float2half_rn((float)(r1 - (double)__half2float(c2)));
        uint16_t *cimg = img + 16384 + (size_t)(64 * hf + n) * 8;
        cimg[0] = __half_as_ushort(c1); cimg[1] = __half_as_ushort(c2); cimg[2] = __half_as_ushort(c3);
      }
      r[TCX_W_FLOATS + 128 + hf] = o.vec_a[k];
    }
  }
}
// RFF record (chisao_tc.cuh, tc_rff_tile): the frequencies cut into three 10-bit fixed-point pieces
// w = 2^(ew-9) (m0 + 2^-10 m1 + 2^-20 m2) (fp64 arithmetic on the fp32 inputs: every step exact), stored as the fp16
// images m0 | m1 | 2^-10 m2, element (n, c) of an image at 16-bit index (c/8)*2048 + n*8 + (c%8); then the constants
void pack_rff_records(const chisao_objective &o, int ew, std::vector<float> &out) {
  out.assign(RFF_REC_FLOATS, 0.0f);
  uint16_t *img = reinterpret_cast<uint16_t *>(out.data());
  const double S0 = std::ldexp(1.0, 9 - ew);
  for (int n = 0; n < o.K; ++n) {
    for (int c = 0; c < o.d; ++c) {
      const double w = (double)o.mats[(size_t)n * o.d + c];
      const double m0 = std::nearbyint(w * S0), r1 = w - m0 / S0;
      const double m1 = std::nearbyint(r1 * S0 * 1024.0), r2 = r1 - m1 / (S0 * 1024.0);
      const double m2 = std::nearbyint(r2 * S0 * 1048576.0);
      const size_t idx = (size_t)(c / 8) * 2048 + (size_t)n * 8 + (c % 8);
      img[idx] = __half_as_ushort(__float2half_rn((float)m0));
      img[8192 + idx] = __half_as_ushort(__float2half_rn((float)m1));
      img[16384 + idx] = __half_as_ushort(__float2half_rn((float)(m2 / 1024.0)));
    }
    float *pr = out.data() + RFF_W_BYTES / 4 + 8 * (n / 2);   // per feature pair: (b0/2pi, b1/2pi, b0, b1) (a0, a1, 0, 0)
    pr[n & 1] = (float)((double)o.vec_b[n] / 6.283185307179586476925);
    pr[2 + (n & 1)] = o.vec_b[n];
    pr[4 + (n & 1)] = o.vec_a[n];
  }
}
// fp16 hi / lo carries 22 bits like tf32 hi / lo as long as nothing overflows (65504) and the lo parts stay above the
// fp16 subnormal spacing 2^-24: max |W| and the box radius (plus the HLC spread) must lie in [2^-3, 2^13]
bool fp16_split_ok(const chisao_objective &o, const chisao_config &c) {
  float wmax = 0.f;
  for (size_t e = 0; e < (size_t)o.K * o.d * o.d; ++e) wmax = std::max(wmax, std::fabs(o.mats[e]));
  const float xmax = eval_point_radius(c);
  const float lo = 0.125f, hi = 8192.0f;
  double cmax = 0.0;                                   // c = W mu goes through the pipe as fp16 pieces as well
  for (int k = 0; k < o.K; ++k)
    for (int n = 0; n < o.d; ++n) {
      double cn = 0.0;
      for (int c2 = 0; c2 < o.d; ++c2) cn += (double)o.mats[((size_t)k * o.d + n) * o.d + c2] * (double)o.means[(size_t)k * o.d + c2];
      cmax = std::max(cmax, std::fabs(cn));
    }
  return wmax >= lo && wmax <= hi && xmax >= lo && xmax <= hi && cmax <= 32768.0 && !getenv("CHISAO_TC_TF32");
}

struct Scope {   // optional CUDA-event bracket around a launch group
  chisao_ctx *c; int cls; cudaEvent_t a = nullptr, b = nullptr;
  Scope(chisao_ctx *ctx, int k) : c(ctx), cls(k) {
    if (!(c->timing & (1u << k))) return;
    auto get = [&]() { cudaEvent_t e; if (!c->pool.empty()) { e = c->pool.back(); c->pool.pop_back(); } else cudaEventCreate(&e); return e; };
    a = get(); b = get();
    cudaEventRecord(a, c->stream);
  }
  ~Scope() {
    if (!a) return;
    cudaEventRecord(b, c->stream);
    c->recs.push_back({cls, a, b});
  }
};

cudaError_t eval_fd(chisao_ctx *c, const float *X, const int32_t *list, const int32_t *count, int mode, float *g_out,
                    int phase, int iter, int counter, int slot_off = 0, int32_t *zero_cnt = nullptr) {
  const State &s = c->st;
  if (s.N == 0) return cudaSuccess;
  FdArgs a{};
  a.X = X; a.list = list; a.count = count; a.max_count = s.N; a.mode = mode; a.d = s.d; a.cycle = c->cycle;
  a.phase = phase; a.iter = iter; a.counter = counter; a.slot_off = slot_off; a.g_out = g_out; a.x = s.x; a.v = s.v; a.lo = s.lo; a.hi = s.hi;
  a.h = c->hp.fd_h; a.mu = c->hp.mu; a.alpha = c->hp.alpha_anti; a.seed = c->hp.seed; a.evals = s.ctrl->evals;
  a.zero_cnt = zero_cnt;
  const int spt = NT / s.d;
  const int grid = (s.N + spt - 1) / spt;
  Scope sc(c, 0);
  c->launches += 1;
  if (c->stencil_aware) return launch_fd_stencil(c->obj, a, s.N, c->stream);   // opt-in, dense objectives only (NEXT-5)
  if (c->use_tc) {
    cudaError_t e = launch_fd_tc(c->obj.id, c->tc, a, s.N, c->stream);
#ifdef CHISAO_DEBUG_SYNC   // debugging builds only: synchronise and report after every tensor-core launch
    fprintf(stderr, "[chisao] fd_tc launched (%s)\n", cudaGetErrorString(e)); e = cudaStreamSynchronize(c->stream); fprintf(stderr, "[chisao] fd_tc done (%s)\n", cudaGetErrorString(e));
#endif
    return e;
  }
  switch (c->obj.id) {
    case 0: return launch_fd_obj_0(c->obj, a, grid, c->stream);
    case 1: return launch_fd_obj_1(c->obj, a, grid, c->stream);
    case 2: return launch_fd_obj_2(c->obj, a, grid, c->stream);
    case 3: return launch_fd_obj_3(c->obj, a, grid, c->stream);
    case 4: return launch_fd_obj_4(c->obj, a, grid, c->stream);
    default: return launch_fd_obj_5(c->obj, a, grid, c->stream);
  }
}

cudaError_t eval_points(chisao_ctx *c, int mode, int b, int iter) {
  const State &s = c->st;
  if (s.N == 0) return cudaSuccess;
  PtArgs a{};
  a.mode = mode; a.b = b; a.d = s.d; a.cycle = c->cycle; a.iter = iter; a.ls_max = c->hp.ls_max; a.max_count = s.N;
  a.f = s.f; a.ft = s.ft; a.dec = s.dec; a.tcur = s.tcur; a.xt = s.xt; a.x = s.x; a.p = s.p; a.g = s.g; a.lo = s.lo; a.hi = s.hi;
  a.ls_b = s.ls_b; a.fd_list = s.fd_list; a.fd_cnt = &s.ctrl->fd_cnt;
  a.c1 = c->hp.ls_c1; a.shrink = c->hp.ls_shrink; a.seed = c->hp.seed; a.evals = s.ctrl->evals;
  if (mode == PT_CENTRE) {
    a.X = s.x; a.list = nullptr; a.count = nullptr;
  } else if (mode == PT_LS_ALL) {
    a.X = s.xt; a.list = s.ls_list[0]; a.count = &s.ctrl->ls_cnt[0];
    // FP32-FMA evaluators at d <= 32: the rows x, p, g of a tile stay in shared memory over the rounds (<= 96 KB more)
    a.rows_in_smem = (!c->use_tc && c->obj.DP <= 32 && eval_smem_bytes(c->obj, ls_rows_bytes(c->obj.DP)) <= 200 * 1024) ? 1 : 0;
  } else {
    a.X = s.xt; a.list = s.ls_list[b % 3]; a.count = &s.ctrl->ls_cnt[b % 3];
    a.next_list = s.ls_list[(b + 1) % 3]; a.next_cnt = &s.ctrl->ls_cnt[(b + 1) % 3];
    a.zero_cnt = &s.ctrl->ls_cnt[(b + 2) % 3];
  }
  const int grid = (s.N + PTILE - 1) / PTILE;
  Scope sc(c, 1);
  c->launches += 1;
  if (c->use_tc) {
    cudaError_t e = launch_pt_tc(c->obj.id, c->tc, a, s.N, c->stream);
#ifdef CHISAO_DEBUG_SYNC
    fprintf(stderr, "[chisao] pt_tc launched (%s)\n", cudaGetErrorString(e)); e = cudaStreamSynchronize(c->stream); fprintf(stderr, "[chisao] pt_tc done (%s)\n", cudaGetErrorString(e));
#endif
    return e;
  }
  switch (c->obj.id) {
    case 0: return launch_pt_obj_0(c->obj, a, grid, c->stream);
    case 1: return launch_pt_obj_1(c->obj, a, grid, c->stream);
    case 2: return launch_pt_obj_2(c->obj, a, grid, c->stream);
    case 3: return launch_pt_obj_3(c->obj, a, grid, c->stream);
    case 4: return launch_pt_obj_4(c->obj, a, grid, c->stream);
    default: return launch_pt_obj_5(c->obj, a, grid, c->stream);
  }
}

cudaError_t hlc_step(chisao_ctx *c, int iter) {
  const State &s = c->st;
  if (s.N == 0) return cudaSuccess;
  HlcArgs a{};
  a.list = s.listE; a.count = &s.ctrl->nE; a.max_count = s.N; a.d = s.d; a.M = s.M; a.cycle = c->cycle; a.iter = iter;
  a.baseline = c->hp.hlc_baseline; a.x = s.x; a.ghat = s.ghat; a.hlc_f = s.hlc_f; a.lo = s.lo; a.hi = s.hi;
  a.sigma_dev = &s.ctrl->sigma_eff; a.eta = c->hp.eta_hlc; a.seed = c->hp.seed; a.evals = s.ctrl->evals;
  const int spt = std::min(PTILE / s.M, HLC_MAX_SPT);
  const int grid = (s.N + spt - 1) / spt;
  Scope sc(c, 2);
  c->launches += 1;
  if (c->use_tc && s.M <= TC_PTS) return launch_hlc_tc(c->obj.id, c->tc, a, s.N, c->stream);
  switch (c->obj.id) {
    case 0: return launch_hlc_obj_0(c->obj, a, grid, c->stream);
    case 1: return launch_hlc_obj_1(c->obj, a, grid, c->stream);
    case 2: return launch_hlc_obj_2(c->obj, a, grid, c->stream);
    case 3: return launch_hlc_obj_3(c->obj, a, grid, c->stream);
    case 4: return launch_hlc_obj_4(c->obj, a, grid, c->stream);
    default: return launch_hlc_obj_5(c->obj, a, grid, c->stream);
  }
}

// ---- units of Algorithm 1 --------------------------------------------------------------------------------
int run_release_eval(chisao_ctx *ctx) {   // Phase 1 start: release all + f, g at x
  // inside a cycle the first L-BFGS iteration's kernel releases (k_lbfgs_step, STEP_FIRST)
  if (!(ctx->in_cycle && ctx->hp.n_conv > 0)) { Scope sc(ctx, 4); CK(launch_release(ctx->st, ctx->stream)); ctx->launches += 1; }
  CK(eval_points(ctx, PT_CENTRE, 0, 0));
  CK(eval_fd(ctx, ctx->st.x, nullptr, nullptr, FD_GRAD, ctx->st.g, 1, 0, EV_INIT));
  return CHISAO_OK;
}
// one L-BFGS iteration (R-4).  As a unit of its own: direction, line search, FD gradient at the accepted
// points, update.  Inside a cycle the update of iteration it - 1 rides in the direction kernel of iteration it (one pass
// over x and g per iteration), and the update of the last iteration (run_lbfgs_finish) also writes Phase 2's partials.
cudaError_t launch_resident(chisao_ctx *c, int it0, int it1, bool diag, bool stick) {
  ResArgs a{};
  a.s = c->st; a.h = c->hp; a.cycle = c->cycle; a.it0 = it0; a.it1 = it1; a.write_diag = diag ? 1 : 0; a.stick_partials = stick ? 1 : 0;
  switch (c->obj.id) {
    case 0: return launch_resident_obj_0(c->obj, a, c->stream);
    case 1: return launch_resident_obj_1(c->obj, a, c->stream);
    case 2: return launch_resident_obj_2(c->obj, a, c->stream);
    case 3: return launch_resident_obj_3(c->obj, a, c->stream);
    case 4: return launch_resident_obj_4(c->obj, a, c->stream);
    default: return launch_resident_obj_5(c->obj, a, c->stream);
  }
}
int run_lbfgs_iter(chisao_ctx *ctx, int it) {
  const State &s = ctx->st;
  if (ctx->resident) {                       // (stand-alone unit; inside a cycle the whole pass is one launch: run_phase1_resident)
    if (s.N == 0) return CHISAO_OK;
    Scope sc(ctx, 0);
    CK(launch_resident(ctx, it, it, true, false));
    ctx->launches += 1;
    return CHISAO_OK;
  }
  const int mode = !ctx->in_cycle ? 0 : (it == 1 ? 1 : 2);
  if (!ctx->in_cycle) CK(cudaMemsetAsync(s.ctrl->ls_cnt, 0, sizeof(int32_t) * 4, ctx->stream));
  { Scope sc(ctx, 3); CK(launch_lbfgs_step(s, ctx->hp, mode, ctx->in_cycle ? it : 0, ctx->stream)); ctx->launches += 1; }
  if (ctx->ls_tile_local) CK(eval_points(ctx, PT_LS_ALL, 0, it));
  else for (int b = 0; b <= ctx->hp.ls_max; ++b) CK(eval_points(ctx, PT_LS, b, it));
  // the FD kernel also zeroes worklist 0's counter for the next iteration's direction kernel
  CK(eval_fd(ctx, s.xt, s.fd_list, &s.ctrl->fd_cnt, FD_GRAD, s.gn, 1, it, EV_LBFGS_FD, 0, &s.ctrl->ls_cnt[0]));
  if (!ctx->in_cycle) { Scope sc(ctx, 4); CK(launch_lbfgs_update(s, ctx->hp, false, ctx->stream)); ctx->launches += 1; }
  return CHISAO_OK;
}
// Phase 1 of a cycle in the history-resident form: release + f, g at the start positions, n_conv iterations and Phase 2's
// partials in one launch
int run_phase1_resident(chisao_ctx *ctx) {
  if (ctx->st.N == 0) return CHISAO_OK;
  CK(cudaMemsetAsync(&ctx->st.ctrl->fmax_enc, 0, sizeof(uint32_t), ctx->stream));
  Scope sc(ctx, 0);
  CK(launch_resident(ctx, 0, ctx->hp.n_conv, false, true));
  ctx->launches += 1;
  return CHISAO_OK;
}
int run_lbfgs_finish(chisao_ctx *ctx) {   // in a cycle: update of the last iteration + ||g||_inf, f_max partials of Phase 2
  Scope sc(ctx, 4);
  CK(launch_lbfgs_update(ctx->st, ctx->hp, true, ctx->stream));
  ctx->launches += 1;
  return CHISAO_OK;
}
int run_stick(chisao_ctx *ctx) {
  Scope sc(ctx, 5);
  // after run_lbfgs_finish the per-sample gradient norms and f_max are already there
  const bool have_partials = ctx->in_cycle && (ctx->hp.n_conv > 0 || ctx->resident);
  CK(launch_stick(ctx->st, ctx->hp, have_partials, ctx->stream));
  ctx->launches += (have_partials ? 0 : 1) + scan_launches(ctx->st.N);
  return CHISAO_OK;
}
int run_dedup(chisao_ctx *ctx) {
  Scope sc(ctx, 5);
  const bool dedup_on = (ctx->hp.phase_mask & (1u << 3)) != 0;
  CK(launch_dedup(ctx->st, ctx->hp, !ctx->in_cycle, ctx->stream));
  ctx->launches += (ctx->in_cycle ? 0 : scan_launches(ctx->st.N)) + (dedup_on ? 1 : 0) + scan_launches(ctx->st.N);
  return CHISAO_OK;
}
int run_reseed(chisao_ctx *ctx) {
  Scope sc(ctx, 6);
  CK(launch_reseed(ctx->st, ctx->hp, ctx->cycle, !ctx->in_cycle, ctx->stream));
  ctx->launches += ctx->in_cycle ? 2 : 3;
  return CHISAO_OK;
}
int run_explore_list(chisao_ctx *ctx) {
  Scope sc(ctx, 5);
  CK(launch_explore_list(ctx->st, ctx->stream));
  ctx->launches += scan_launches(ctx->st.N);
  return CHISAO_OK;
}
int run_hlc(chisao_ctx *ctx, int t) {
  if (!(ctx->hp.phase_mask & (1u << 5))) return CHISAO_OK;
  if (!(ctx->hp.sigma_s > 0.0f)) { Scope sc(ctx, 2); CK(launch_hlc_sigma(ctx->st, ctx->hp, ctx->stream)); ctx->launches += 2; }
  if (ctx->hp.hlc_baseline == 2) {   // the paper's Eq. 5 form: K FD gradients at perturbed points (NEXT-2)
    const State &s = ctx->st;
    for (int k = 0; k < ctx->hp.hlc_M; ++k) {
      { Scope sc(ctx, 2); CK(launch_hlc5(s, ctx->hp, ctx->cycle, t, k, 0, ctx->stream)); ctx->launches += 1; }
      CK(eval_fd(ctx, s.xt, s.listE, &s.ctrl->nE, FD_GRAD, s.gn, 5, t, EV_HLC, k * 2 * s.d));
      { Scope sc(ctx, 2); CK(launch_hlc5(s, ctx->hp, ctx->cycle, t, k, 1, ctx->stream)); ctx->launches += 1; }
    }
    { Scope sc(ctx, 2); CK(launch_hlc5(s, ctx->hp, ctx->cycle, t, 0, 2, ctx->stream)); ctx->launches += 1; }
    return CHISAO_OK;
  }
  CK(hlc_step(ctx, t));
  return CHISAO_OK;
}
int run_anti(chisao_ctx *ctx, int t) {
  if (!(ctx->hp.phase_mask & (1u << 6))) return CHISAO_OK;
  const State &s = ctx->st;
  CK(eval_fd(ctx, s.x, s.listE, &s.ctrl->nE, FD_ANTI, nullptr, 6, t, EV_ANTI));
  return CHISAO_OK;
}

int read_stats(chisao_ctx *ctx, chisao_stats *out) {
  Ctrl h;
  CK(cudaMemcpyAsync(&h, ctx->st.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  out->cycle = ctx->cycle; out->n_stuck = h.n_stuck; out->k_lost = h.k_lost; out->n_active = h.n_active;
  out->reseed_strategy = h.strategy; out->gr_enabled = h.gr_enabled;
  for (int k = 0; k < 8; ++k) out->evals[k] = h.evals[k];
  out->f_max = dec_ordered(h.fmax_enc);
  return CHISAO_OK;
}

}  // namespace

extern "C" {

int chisao_workspace_bytes(const chisao_config *cfg, const chisao_objective *obj, size_t *bytes) {
  std::string why;
  const int rc = validate(cfg, obj, why);
  if (rc) return fail(nullptr, rc, why);
  if (!bytes) return fail(nullptr, CHISAO_E_INVALID, "bytes is null");
  *bytes = carve(*cfg, *obj, nullptr, nullptr, nullptr);
  return CHISAO_OK;
}

int chisao_init(chisao_ctx **out, const chisao_config *cfg, const chisao_objective *obj, float *x_dev,
                void *workspace_dev, size_t workspace_bytes, void *stream) {
  std::string why;
  int rc = validate(cfg, obj, why);
  if (rc) return fail(nullptr, rc, why);
  if (!out) return fail(nullptr, CHISAO_E_INVALID, "out is null");
  if (cfg->N > 0 && !x_dev) return fail(nullptr, CHISAO_E_INVALID, "x_dev is null");
  const size_t need = carve(*cfg, *obj, nullptr, nullptr, nullptr);
  if (!workspace_dev || workspace_bytes < need) return fail(nullptr, CHISAO_E_WORKSPACE, "workspace too small");
  if (reinterpret_cast<uintptr_t>(workspace_dev) & 255) return fail(nullptr, CHISAO_E_WORKSPACE, "workspace not 256-byte aligned");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) return cuda_fail(nullptr, e == cudaSuccess ? cudaErrorNoDevice : e, "no CUDA device");

  chisao_ctx *ctx = new chisao_ctx();
  ctx->cfg = *cfg;
  ctx->stream = reinterpret_cast<cudaStream_t>(stream);
  ctx->ws_bytes = need;
  ctx->lo.assign(cfg->lo, cfg->lo + cfg->d);
  ctx->hi.assign(cfg->hi, cfg->hi + cfg->d);
  ctx->cfg.lo = ctx->lo.data(); ctx->cfg.hi = ctx->hi.data();
  Hyper &h = ctx->hp;
  h.n_osc = cfg->n_osc; h.n_conv = cfg->n_conv; h.n_anti = cfg->n_anti; h.n_cloud = cfg->n_cloud; h.hlc_M = cfg->hlc_M;
  h.lbfgs_m = cfg->lbfgs_m; h.ls_max = cfg->ls_max; h.reseed_cands = cfg->reseed_cands; h.hlc_baseline = cfg->hlc_baseline;
  h.phase_mask = cfg->phase_mask; h.fd_h = cfg->fd_h; h.eps_grad = cfg->eps_grad; h.eps_dup = cfg->eps_dup;
  h.log_delta = cfg->log_delta; h.mu = cfg->mu; h.alpha_anti = cfg->alpha_anti; h.eta_hlc = cfg->eta_hlc;
  h.sigma_s = cfg->sigma_s; h.ls_c1 = cfg->ls_c1; h.ls_shrink = cfg->ls_shrink; h.seed = cfg->seed;

  State &s = ctx->st;
  std::memset(&s, 0, sizeof(s));
  s.N = cfg->N; s.d = cfg->d; s.m = cfg->lbfgs_m; s.M = cfg->hlc_M; s.x = x_dev;
  const float *recs_dev = nullptr, *tc_dev = nullptr;
  carve(*cfg, *obj, static_cast<unsigned char *>(workspace_dev), &s, &recs_dev, &tc_dev);

  DevObj &o = ctx->obj;
  o.id = obj->id; o.d = obj->d; o.K = obj->K; o.DP = padded_dim(obj->d);
  o.rec = record_floats(o.id, o.DP);
  o.kc = std::max(1, std::min(o.K, CHUNK_BYTES / (o.rec * 4)));
  o.sigma_noise = obj->sigma_noise;
  o.recs = recs_dev;
  pack_records(*obj, o.DP, ctx->recs_host, o.s0);
  if (eval_smem_bytes(o, hlc_extra_bytes(o.DP)) > 200 * 1024) {
    delete ctx;
    return fail(nullptr, CHISAO_E_INVALID, "objective record too large for shared memory");
  }

#define CKI(call)                                                                   \
  do {                                                                              \
    cudaError_t e_ = (call);                                                        \
    if (e_ != cudaSuccess) { int r_ = cuda_fail(nullptr, e_, #call); delete ctx; return r_; } \
  } while (0)
  switch (o.id) {
    case 0: CKI(configure_obj_0()); break;
    case 1: CKI(configure_obj_1()); break;
    case 2: CKI(configure_obj_2()); break;
    case 3: CKI(configure_obj_3()); break;
    case 4: CKI(configure_obj_4()); break;
    default: CKI(configure_obj_5()); break;
  }
  ctx->use_tc = wants_tc(*obj, *cfg);
  if (ctx->use_tc) {
    ctx->tc.f16 = (obj->id == CHISAO_OBJ_GMM_FULL && fp16_split_ok(*obj, *cfg)) ? 1 : 0;
    ctx->tc.quad_ws = 0;
    if (obj->id == CHISAO_OBJ_QUAD) { int ws = 0; if (quad16_scale(*obj, &ws)) { ctx->tc.f16 = 1; ctx->tc.quad_ws = ws; } }
    if (obj->id == CHISAO_OBJ_RFF) {
      int ex = 0, ew = 0;
      rff_tc_scales(*obj, *cfg, &ex, &ew);
      pack_rff_records(*obj, ew, ctx->tc_host);
      ctx->tc.rff_S0 = std::ldexp(1.0f, 9 - ex); ctx->tc.rff_uA = std::ldexp(1.0f, ex + ew - 18);
      ctx->tc.rff_s0 = obj->scalar0; ctx->tc.nchunk = (obj->K + 63) / 64;
      const double uA = std::ldexp(1.0, ex + ew - 18), P = 6.283185307179586476925 / uA, Phi = std::nearbyint(P);
      ctx->tc.rff_cA = (float)(uA / 6.283185307179586476925); ctx->tc.rff_Phi = (float)Phi; ctx->tc.rff_cL = (float)(-(P - Phi) * uA);
    } else if (ctx->tc.f16 && obj->id == CHISAO_OBJ_QUAD) pack_quad16_record(*obj, ctx->tc.quad_ws, ctx->tc_host);
    else if (ctx->tc.f16) pack_tcx16_records(*obj, ctx->tc_host);
    else if (obj->id == CHISAO_OBJ_GMM_FULL) pack_tcx_records(*obj, ctx->tc_host);
    else pack_tc_records(*obj, ctx->tc_host);
    ctx->tc.npair = (obj->K + 1) / 2;
    ctx->tc.K = obj->K; ctx->tc.d = obj->d; ctx->tc.sigma_noise = obj->sigma_noise; ctx->tc.recs = tc_dev;
    CKI(tc_configure());
  }
  {   // line search form (see chisao_ctx::ls_tile_local): plain-definition flop per evaluation as the cost of a tile
    const double dd = obj->d, KK = obj->K;
    double cost = 0.0;
    switch (obj->id) {
      case CHISAO_OBJ_GMM_ISO: cost = KK * 3 * dd; break;
      case CHISAO_OBJ_GMM_DIAG: cost = KK * 4 * dd; break;
      case CHISAO_OBJ_GMM_FULL: cost = KK * 2 * dd * dd; break;
      case CHISAO_OBJ_RFF: cost = KK * 4 * dd; break;      // fp64 phases at half rate on the FP32-FMA evaluator
      case CHISAO_OBJ_QUAD: cost = 2 * dd * dd; break;
      default: cost = 64 * dd; break;                      // Appendix-D functions
    }
    ctx->ls_tile_local = ctx->use_tc ? (obj->id != CHISAO_OBJ_GMM_FULL) : (cost <= 32768.0);
    if (getenv("CHISAO_LS_PER_TRIAL")) ctx->ls_tile_local = false;
    const int dd_ = obj->d;
    ctx->resident_ok = !ctx->use_tc && dd_ <= 32 && (dd_ & (dd_ - 1)) == 0 && o.kc >= o.K && cfg->lbfgs_m <= 16 &&
                       eval_smem_bytes(o, resident_extra_bytes()) <= 200 * 1024;
    ctx->resident = ctx->resident_ok && !getenv("CHISAO_LBFGS_SPILL");
    if (ctx->resident_ok) {
      switch (o.id) {
        case 0: CKI(configure_resident_obj_0()); break;
        case 1: CKI(configure_resident_obj_1()); break;
        case 2: CKI(configure_resident_obj_2()); break;
        case 3: CKI(configure_resident_obj_3()); break;
        case 4: CKI(configure_resident_obj_4()); break;
        default: CKI(configure_resident_obj_5()); break;
      }
    }
  }
  // zero everything except the parameter records, then upload parameters and bounds
  CKI(cudaMemsetAsync(workspace_dev, 0, need, ctx->stream));
  CKI(cudaMemcpyAsync(const_cast<float *>(recs_dev), ctx->recs_host.data(), ctx->recs_host.size() * 4,
                      cudaMemcpyHostToDevice, ctx->stream));
  if (ctx->use_tc)
    CKI(cudaMemcpyAsync(const_cast<float *>(tc_dev), ctx->tc_host.data(), ctx->tc_host.size() * 4, cudaMemcpyHostToDevice,
                        ctx->stream));
  CKI(cudaMemcpyAsync(s.lo, ctx->lo.data(), 4 * (size_t)cfg->d, cudaMemcpyHostToDevice, ctx->stream));
  CKI(cudaMemcpyAsync(s.hi, ctx->hi.data(), 4 * (size_t)cfg->d, cudaMemcpyHostToDevice, ctx->stream));
  const int32_t one = 1;
  CKI(cudaMemcpyAsync(&s.ctrl->gr_enabled, &one, 4, cudaMemcpyHostToDevice, ctx->stream));
  if (cfg->sigma_s > 0.0f)   // caller-supplied smoothing scale: constant for the life of the context
    CKI(cudaMemcpyAsync(&s.ctrl->sigma_eff, &ctx->hp.sigma_s, 4, cudaMemcpyHostToDevice, ctx->stream));
#undef CKI
  *out = ctx;
  return CHISAO_OK;
}

int chisao_seed_population(chisao_ctx *ctx) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  CK(launch_seed_population(ctx->st, ctx->hp, ctx->stream));
  ctx->launches += 1;
  return CHISAO_OK;
}

// the launch sequence of one cycle k = ctx->cycle on ctx->stream (Algorithm 1)
static int enqueue_cycle_units(chisao_ctx *ctx);
static int enqueue_cycle(chisao_ctx *ctx) {
  ctx->in_cycle = true;
  const int rc = enqueue_cycle_units(ctx);
  ctx->in_cycle = false;
  return rc;
}
static int enqueue_cycle_units(chisao_ctx *ctx) {
  int rc;
  if (ctx->resident) {
    if ((rc = run_phase1_resident(ctx))) return rc;   // Phase 1 in one launch, history in registers
  } else {
    if ((rc = run_release_eval(ctx))) return rc;      // Phase 1: release all, then converge
    for (int it = 1; it <= ctx->hp.n_conv; ++it)
      if ((rc = run_lbfgs_iter(ctx, it))) return rc;
    if (ctx->hp.n_conv > 0 && (rc = run_lbfgs_finish(ctx))) return rc;
  }
  if ((rc = run_stick(ctx))) return rc;               // Phase 2
  if ((rc = run_dedup(ctx))) return rc;               // Phase 3 (its list kernel also clears ctrl->strategy)
  if (ctx->cycle < ctx->hp.n_osc) {                   // "if k < n_osc"
    if ((rc = run_reseed(ctx))) return rc;            // Phase 4
    if ((rc = run_explore_list(ctx))) return rc;
    for (int t = 1; t <= ctx->hp.n_cloud; ++t)        // Phase 5
      if ((rc = run_hlc(ctx, t))) return rc;
    for (int t = 1; t <= ctx->hp.n_anti; ++t)         // Phase 6
      if ((rc = run_anti(ctx, t))) return rc;
  }
  return CHISAO_OK;
}

// The same sequence submitted as ONE graph launch: every launch already reads its counts from the device control
// block, so the sequence is static; only the cycle index (a kernel argument) changes, hence capture + ExecUpdate per
// cycle (host cost ~1 us per node instead of a launch each; the GPU runs the nodes back to back).  Any failure of the
// graph machinery switches it off for the context and the cycle is submitted directly.
static int step_graph(chisao_ctx *ctx) {
  cudaStream_t user = ctx->stream;
  auto give_up = [&]() { ctx->graph_on = false; cudaGetLastError(); return enqueue_cycle(ctx); };
  if (!ctx->gstream) {
    if (cudaStreamCreateWithFlags(&ctx->gstream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->gfork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->gjoin, cudaEventDisableTiming) != cudaSuccess)
      return give_up();
  }
  if (cudaStreamBeginCapture(ctx->gstream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) return give_up();
  ctx->stream = ctx->gstream;
  const uint64_t l0 = ctx->launches;
  const int rc = enqueue_cycle(ctx);
  ctx->stream = user;
  cudaGraph_t graph = nullptr;
  const cudaError_t ec = cudaStreamEndCapture(ctx->gstream, &graph);
  if (rc || ec != cudaSuccess || !graph) {
    if (graph) cudaGraphDestroy(graph);
    ctx->launches = l0;
    if (rc) { ctx->graph_on = false; cudaGetLastError(); return rc; }
    return give_up();
  }
  const int slot = ctx->cycle < ctx->hp.n_osc ? 0 : 1;
  if (ctx->gexec[slot]) {
    cudaGraphExecUpdateResultInfo info;
    if (cudaGraphExecUpdate(ctx->gexec[slot], graph, &info) != cudaSuccess) {
      cudaGetLastError();
      cudaGraphExecDestroy(ctx->gexec[slot]);
      ctx->gexec[slot] = nullptr;
    }
  }
  if (!ctx->gexec[slot] && cudaGraphInstantiate(&ctx->gexec[slot], graph, 0) != cudaSuccess) {
    ctx->gexec[slot] = nullptr;
    cudaGraphDestroy(graph);
    ctx->launches = l0;
    return give_up();
  }
  cudaGraphDestroy(graph);
  CK(cudaEventRecord(ctx->gfork, user));
  CK(cudaStreamWaitEvent(ctx->gstream, ctx->gfork, 0));
  CK(cudaGraphLaunch(ctx->gexec[slot], ctx->gstream));
  CK(cudaEventRecord(ctx->gjoin, ctx->gstream));
  CK(cudaStreamWaitEvent(user, ctx->gjoin, 0));
  ctx->graph_launches += 1;
  return CHISAO_OK;
}

int chisao_step(chisao_ctx *ctx, chisao_stats *stats) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  if (ctx->cycle >= ctx->hp.n_osc) return fail(ctx, CHISAO_E_STATE, "all n_osc cycles already done");
  ctx->cycle += 1;                                    // "for k = 1..n_osc"
  // per-launch event bracketing (chisao_timing_enable) needs the launches on the stream itself
#ifdef CHISAO_DEBUG_SYNC
  const bool graph = false;
#else
  const bool graph = ctx->graph_on && ctx->timing == 0 && ctx->st.N > 0;
#endif
  const int rc = graph ? step_graph(ctx) : enqueue_cycle(ctx);
  if (rc) { ctx->cycle -= 1; return rc; }             // a cycle that could not be enqueued does not advance k (nor the Philox keys)
  if (stats) return read_stats(ctx, stats);
  return CHISAO_OK;
}

int chisao_step_host(chisao_ctx *ctx, const float *x_in, float *x_out, float *f_out, uint8_t *stuck_out,
                     chisao_stats *stats) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  const size_t N = ctx->st.N, d = ctx->st.d;
  if (x_in) CK(cudaMemcpyAsync(ctx->st.x, x_in, N * d * 4, cudaMemcpyHostToDevice, ctx->stream));
  const int rc = chisao_step(ctx, nullptr);
  if (rc) return rc;
  if (x_out) CK(cudaMemcpyAsync(x_out, ctx->st.x, N * d * 4, cudaMemcpyDeviceToHost, ctx->stream));
  if (f_out) CK(cudaMemcpyAsync(f_out, ctx->st.f, N * 4, cudaMemcpyDeviceToHost, ctx->stream));
  if (stuck_out) CK(cudaMemcpyAsync(stuck_out, ctx->st.stuck, N, cudaMemcpyDeviceToHost, ctx->stream));
  if (stats) return read_stats(ctx, stats);
  CK(cudaStreamSynchronize(ctx->stream));
  return CHISAO_OK;
}

int chisao_phase(chisao_ctx *ctx, int32_t phase_id, int32_t iter) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  switch (phase_id) {
    case CHISAO_PH_RELEASE_EVAL: return run_release_eval(ctx);
    case CHISAO_PH_LBFGS_ITER: return run_lbfgs_iter(ctx, iter);
    case CHISAO_PH_LBFGS_DIRECTION: {
      CK(cudaMemsetAsync(ctx->st.ctrl->ls_cnt, 0, sizeof(int32_t) * 4, ctx->stream));
      Scope sc(ctx, 3);
      CK(launch_lbfgs_step(ctx->st, ctx->hp, 0, 0, ctx->stream));
      ctx->launches += 1;
      return CHISAO_OK;
    }
    case CHISAO_PH_STICK: return run_stick(ctx);
    case CHISAO_PH_DEDUP: return run_dedup(ctx);
    case CHISAO_PH_RESEED: return run_reseed(ctx);
    case CHISAO_PH_HLC_STEP: { const int rc = run_explore_list(ctx); return rc ? rc : run_hlc(ctx, iter); }
    case CHISAO_PH_ANTI_STEP: { const int rc = run_explore_list(ctx); return rc ? rc : run_anti(ctx, iter); }
  }
  return fail(ctx, CHISAO_E_INVALID, "unknown phase id");
}

int chisao_get_stats(chisao_ctx *ctx, chisao_stats *stats) {
  if (!ctx || !stats) return fail(ctx, CHISAO_E_INVALID, "null argument");
  return read_stats(ctx, stats);
}

int chisao_modes(chisao_ctx *ctx, float *modes_out, float *f_out, int32_t *idx_out, int32_t cap, int32_t *n_modes) {
  if (!ctx || !n_modes || cap < 0) return fail(ctx, CHISAO_E_INVALID, "bad argument");
  const State &s = ctx->st;
  const size_t N = s.N, d = s.d;
  std::vector<uint8_t> stuck(N);
  std::vector<float> f(N);
  if (N) {
    CK(cudaMemcpyAsync(stuck.data(), s.stuck, N, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaMemcpyAsync(f.data(), s.f, N * 4, cudaMemcpyDeviceToHost, ctx->stream));
  }
  CK(cudaStreamSynchronize(ctx->stream));
  std::vector<int32_t> idx;
  for (size_t i = 0; i < N; ++i) if (stuck[i]) idx.push_back((int32_t)i);
  std::stable_sort(idx.begin(), idx.end(), [&](int32_t a, int32_t b) { return f[a] > f[b]; });  // (f desc, index asc)
  *n_modes = (int32_t)idx.size();
  const int n = std::min<int>(cap, (int)idx.size());
  if (n > 0) {
    if (modes_out) {   // gather on the device (gn and fd_list are free between cycles)
      CK(cudaMemcpyAsync(s.fd_list, idx.data(), (size_t)n * 4, cudaMemcpyHostToDevice, ctx->stream));
      CK(launch_gather_rows(s.x, s.fd_list, n, (int)d, s.gn, ctx->stream));
      ctx->launches += 1;
      CK(cudaMemcpyAsync(modes_out, s.gn, (size_t)n * d * 4, cudaMemcpyDeviceToHost, ctx->stream));
      CK(cudaStreamSynchronize(ctx->stream));
    }
    for (int q = 0; q < n; ++q) {
      if (f_out) f_out[q] = f[idx[q]];
      if (idx_out) idx_out[q] = idx[q];
    }
  }
  if ((int)idx.size() > cap) return fail(ctx, CHISAO_E_CAPACITY, "cap < n_modes");
  return CHISAO_OK;
}

static int field_info(chisao_ctx *ctx, int32_t field, void **dev, size_t *bytes) {
  const State &s = ctx->st;
  const size_t N = s.N, d = s.d, M = s.M;
  switch (field) {
    case CHISAO_X: *dev = s.x; *bytes = N * d * 4; return 0;
    case CHISAO_F: *dev = s.f; *bytes = N * 4; return 0;
    case CHISAO_G: *dev = s.g; *bytes = N * d * 4; return 0;
    case CHISAO_V: *dev = s.v; *bytes = N * d * 4; return 0;
    case CHISAO_STUCK: *dev = s.stuck; *bytes = N; return 0;
    case CHISAO_REMOVED: *dev = s.removed; *bytes = N; return 0;
    case CHISAO_STALLED: *dev = s.stalled; *bytes = N; return 0;
    case CHISAO_HIST_LEN: *dev = s.hist_len; *bytes = N * 4; return 0;
    case CHISAO_P: *dev = s.p; *bytes = N * d * 4; return 0;
    case CHISAO_LS_B: *dev = s.ls_b; *bytes = N * 4; return 0;
    case CHISAO_GHAT: *dev = s.ghat; *bytes = N * d * 4; return 0;
    case CHISAO_HLC_F: *dev = s.hlc_f; *bytes = N * M * 4; return 0;
    case CHISAO_RS_SRC: *dev = s.rs_src; *bytes = N * 4; return 0;
    case CHISAO_RS_CAND: *dev = s.rs_cand; *bytes = N * 4; return 0;
    case CHISAO_XT: *dev = s.xt; *bytes = N * d * 4; return 0;
    case CHISAO_GR_Q: *dev = s.grQ; *bytes = d * d * 4; return 0;
    case CHISAO_SIGMA: *dev = &s.ctrl->sigma_eff; *bytes = 4; return 0;
  }
  return -1;
}

int chisao_get_state(chisao_ctx *ctx, int32_t field, void *dst, size_t bytes) {
  if (!ctx || (!dst && bytes)) return fail(ctx, CHISAO_E_INVALID, "null argument");
  const State &s = ctx->st;
  const size_t N = s.N, d = s.d, m = s.m;
  if (field == CHISAO_CTRL) {
    if (bytes != 32) return fail(ctx, CHISAO_E_INVALID, "CTRL is 8 x i32");
    Ctrl h;
    CK(cudaMemcpyAsync(&h, s.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    int32_t c[8] = {ctx->cycle, h.gr_enabled, h.gr_unproductive, h.gr_prev_modes, h.gr_used_last, h.k_lost, h.n_stuck, h.n_active};
    std::memcpy(dst, c, 32);
    return CHISAO_OK;
  }
  if (field == CHISAO_HIST_S || field == CHISAO_HIST_Y) {
    if (bytes != m * N * d * 4) return fail(ctx, CHISAO_E_INVALID, "wrong size for history field");
    std::vector<float> phys(m * N * d);
    std::vector<int32_t> head(N), len(N);
    if (N) {
      CK(cudaMemcpy2DAsync(phys.data(), N * d * 4, field == CHISAO_HIST_S ? s.S : s.Y, s.hplane * 4, N * d * 4, m, cudaMemcpyDeviceToHost, ctx->stream));
      CK(cudaMemcpyAsync(head.data(), s.hist_head, N * 4, cudaMemcpyDeviceToHost, ctx->stream));
      CK(cudaMemcpyAsync(len.data(), s.hist_len, N * 4, cudaMemcpyDeviceToHost, ctx->stream));
    }
    CK(cudaStreamSynchronize(ctx->stream));
    float *o = static_cast<float *>(dst);
    std::memset(o, 0, bytes);
    for (size_t i = 0; i < N; ++i)
      for (int l = 0; l < len[i]; ++l) {
        const size_t ph = (size_t)(head[i] + l) % m;
        std::memcpy(o + ((size_t)l * N + i) * d, phys.data() + (ph * N + i) * d, d * 4);
      }
    return CHISAO_OK;
  }
  void *dev = nullptr; size_t fb = 0;
  if (field_info(ctx, field, &dev, &fb)) return fail(ctx, CHISAO_E_INVALID, "unknown state field");
  if (fb != bytes) return fail(ctx, CHISAO_E_INVALID, "wrong size for state field");
  if (bytes) CK(cudaMemcpyAsync(dst, dev, bytes, cudaMemcpyDeviceToHost, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  return CHISAO_OK;
}

int chisao_set_state(chisao_ctx *ctx, int32_t field, const void *src, size_t bytes) {
  if (!ctx || (!src && bytes)) return fail(ctx, CHISAO_E_INVALID, "null argument");
  const State &s = ctx->st;
  const size_t N = s.N, d = s.d, m = s.m;
  if (field == CHISAO_CTRL) {
    if (bytes != 32) return fail(ctx, CHISAO_E_INVALID, "CTRL is 8 x i32");
    int32_t c[8];
    std::memcpy(c, src, 32);
    ctx->cycle = c[0];
    CK(cudaMemcpyAsync(&s.ctrl->cycle, c, 32, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return CHISAO_OK;
  }
  if (field == CHISAO_HIST_S || field == CHISAO_HIST_Y) {
    // logical order in, physical = logical: ring heads are reset (set HIST_S, HIST_Y and HIST_LEN together)
    if (bytes != m * N * d * 4) return fail(ctx, CHISAO_E_INVALID, "wrong size for history field");
    if (bytes) {
      CK(cudaMemcpy2DAsync(field == CHISAO_HIST_S ? s.S : s.Y, s.hplane * 4, src, N * d * 4, N * d * 4, m, cudaMemcpyHostToDevice, ctx->stream));
      CK(cudaMemsetAsync(s.hist_head, 0, N * 4, ctx->stream));
    }
    CK(cudaStreamSynchronize(ctx->stream));
    return CHISAO_OK;
  }
  if (field >= CHISAO_P) return fail(ctx, CHISAO_E_INVALID, "diagnostic fields are read-only");
  void *dev = nullptr; size_t fb = 0;
  if (field_info(ctx, field, &dev, &fb)) return fail(ctx, CHISAO_E_INVALID, "unknown state field");
  if (fb != bytes) return fail(ctx, CHISAO_E_INVALID, "wrong size for state field");
  if (bytes) CK(cudaMemcpyAsync(dev, src, bytes, cudaMemcpyHostToDevice, ctx->stream));
  CK(cudaStreamSynchronize(ctx->stream));
  return CHISAO_OK;
}

int chisao_set_option(chisao_ctx *ctx, int32_t option, int32_t value) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  if (option == CHISAO_OPT_STENCIL_AWARE) {
    if (value && !fd_stencil_supported(ctx->obj))
      return fail(ctx, CHISAO_E_INVALID, "the stencil-aware FD evaluator exists for GMM_FULL and QUAD only");
    ctx->stencil_aware = value != 0;
    return CHISAO_OK;
  }
  if (option == CHISAO_OPT_CUDA_GRAPH) { ctx->graph_on = value != 0; return CHISAO_OK; }
  if (option == CHISAO_OPT_LBFGS_RESIDENT) {
    if (value && !ctx->resident_ok)
      return fail(ctx, CHISAO_E_INVALID, "the history-resident L-BFGS pass needs an FP32-FMA evaluator, d in {1,2,4,8,16,32}, parameters in one chunk, m <= 16");
    ctx->resident = value != 0;
    for (auto &ge : ctx->gexec) if (ge) { cudaGraphExecDestroy(ge); ge = nullptr; }   // another topology
    return CHISAO_OK;
  }
  if (option == CHISAO_OPT_LS_TILE_LOCAL) {
    if (value && ctx->use_tc && ctx->obj.id == CHISAO_OBJ_GMM_FULL)
      return fail(ctx, CHISAO_E_INVALID, "the tile-local line search does not exist for the x-stationary GMM_FULL evaluator");
    ctx->ls_tile_local = value != 0;
    for (auto &ge : ctx->gexec) if (ge) { cudaGraphExecDestroy(ge); ge = nullptr; }   // another topology
    return CHISAO_OK;
  }
  return fail(ctx, CHISAO_E_INVALID, "unknown option");
}

int chisao_get_info(const chisao_ctx *ctx, int32_t which, int32_t *value) {
  if (ctx && value && which == CHISAO_INFO_GRAPH_LAUNCHES) { *value = (int32_t)ctx->graph_launches; return CHISAO_OK; }
  if (ctx && value && which == CHISAO_INFO_LS_TILE_LOCAL) { *value = ctx->ls_tile_local ? 1 : 0; return CHISAO_OK; }
  if (ctx && value && which == CHISAO_INFO_LBFGS_RESIDENT) { *value = ctx->resident ? 1 : 0; return CHISAO_OK; }
  if (!ctx || !value || which != CHISAO_INFO_EVALUATOR) return CHISAO_E_INVALID;
  *value = !ctx->use_tc ? 0 : (ctx->obj.id == CHISAO_OBJ_RFF ? 4 : (ctx->obj.id == CHISAO_OBJ_QUAD ? (ctx->tc.f16 ? 5 : 1) : (ctx->tc.f16 ? 3 : 2)));
  return CHISAO_OK;
}

uint64_t chisao_launch_count(const chisao_ctx *ctx) { return ctx ? ctx->launches : 0; }

int chisao_timing_enable(chisao_ctx *ctx, int32_t on) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  ctx->timing = on == 1 ? 0xFFFFFFFFu : (on <= 0 ? 0u : ((uint32_t)on >> 1));   // 1: every class; else bit k + 1 selects class k
  return CHISAO_OK;
}
int chisao_timing_reset(chisao_ctx *ctx) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  CK(cudaStreamSynchronize(ctx->stream));
  for (auto &r : ctx->recs) { ctx->pool.push_back(r.a); ctx->pool.push_back(r.b); }
  ctx->recs.clear();
  return CHISAO_OK;
}
int chisao_timing_get(chisao_ctx *ctx, int32_t which, double *ms, uint64_t *launches) {
  if (!ctx) return fail(nullptr, CHISAO_E_INVALID, "null ctx");
  CK(cudaStreamSynchronize(ctx->stream));
  double tot = 0.0; uint64_t n = 0;
  for (auto &r : ctx->recs) {
    if (r.cls != which) continue;
    float t = 0.f;
    CK(cudaEventElapsedTime(&t, r.a, r.b));
    tot += t; n += 1;
  }
  if (ms) *ms = tot;
  if (launches) *launches = n;
  return CHISAO_OK;
}

const char *chisao_last_error(const chisao_ctx *ctx) { return ctx ? ctx->err.c_str() : g_last_error.c_str(); }

void chisao_destroy(chisao_ctx *ctx) {
  if (!ctx) return;
  for (auto &r : ctx->recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto &e : ctx->pool) cudaEventDestroy(e);
  for (auto &ge : ctx->gexec) if (ge) cudaGraphExecDestroy(ge);
  if (ctx->gfork) cudaEventDestroy(ctx->gfork);
  if (ctx->gjoin) cudaEventDestroy(ctx->gjoin);
  if (ctx->gstream) cudaStreamDestroy(ctx->gstream);
  delete ctx;
}

}  // extern "C"
