// chisao_select.cu -- Phases 2-4: stick test (Eq. 3), L-infinity deduplication (Eq. 4),
// ascending index lists by an ordered block scan, Golden-Rooster bookkeeping, and reseeding
// (Repulse Monkey / Golden Rooster / uniform refill).  Readings R-7..R-10, R-13.
#include "chisao_device.cuh"

namespace chisao {

constexpr int SCAN_BLOCK = 1024;   // samples per scan block (one per thread)

// ---- Phase 2 (Eq. 3): ||grad f||_inf per sample and f_max = max_i f(x_i) (Alg. 1, R-13) ---
__global__ void __launch_bounds__(256) k_ginf_fmax(State s) {
  __shared__ float sh_max[8];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int i = blockIdx.x * 8 + wib;
  float fm = -INFINITY;
  if (i < s.N) {
    const float *g = s.g + (size_t)i * s.d;
    float gi = 0.0f;
    bool nan = false;
    for (int j = lane; j < s.d; j += 32) { const float a = fabsf(g[j]); nan |= !(a == a); gi = fmaxf(gi, a); }
    gi = warp_max(gi);
    nan = __any_sync(0xffffffffu, nan);
    if (lane == 0) {
      s.ginf[i] = nan ? NAN : gi;    // a NaN gradient can never pass "< eps_grad"
      const float f = s.f[i];
      if (fabsf(f) <= 3.0e38f) fm = f;   // finite values only
    }
  }
  if (lane == 0) sh_max[wib] = fm;
  __syncthreads();
  if (threadIdx.x == 0) {
    float mx = sh_max[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) mx = fmaxf(mx, sh_max[w]);
    if (mx > -INFINITY) atomicMax(&s.ctrl->fmax_enc, enc_ordered(mx));
  }
}

// stuck_i = (||grad f(x_i)||_inf < eps_grad) and (f(x_i) >= f_max + log delta)   (Eq. 3)
__device__ __forceinline__ bool stick_test(const State &s, const Hyper &h, int i) {
  const float fmax = dec_ordered(s.ctrl->fmax_enc);
  const float f = s.f[i];
  return (s.ginf[i] < h.eps_grad) && (fabsf(f) <= 3.0e38f) && (f >= fmax + h.log_delta);
}

// ---- ordered compaction: ascending index lists by class ------------------------------------------------
// SCAN_STICK  : class 1 = stuck                         -> listP0
// SCAN_STICK_FLAGS: the same, and the counting kernel first WRITES the flags of Eq. 3 (stuck, removed <- 0)
// SCAN_FINAL  : class 0 = unfrozen (not stuck, not removed) -> listA, 1 = stuck -> listP, 2 = removed -> listR; the
//               counting kernel clears the stuck flag of removed samples ("removed" in Eq. 4 means it no longer is a mode),
//               the scatter kernel resets the reseed diagnostics
// SCAN_EXPLORE: class 1 = not stuck and not removed     -> listE
__device__ __forceinline__ int scan_class(const State &s, int mode, int i) {
  const bool st = s.stuck[i] != 0, rm = s.removed[i] != 0;
  if (mode == SCAN_STICK || mode == SCAN_STICK_FLAGS) return st ? 1 : -1;
  if (mode == SCAN_EXPLORE) return (!st && !rm) ? 1 : -1;
  return rm ? 2 : (st ? 1 : 0);
}

__global__ void __launch_bounds__(SCAN_BLOCK) k_scan_count(State s, Hyper h, int mode, int nb) {
  __shared__ int cnt[3];
  if (threadIdx.x < 3) cnt[threadIdx.x] = 0;
  __syncthreads();
  const int i = blockIdx.x * SCAN_BLOCK + threadIdx.x;
  if (i < s.N) {
    if (mode == SCAN_STICK_FLAGS) { s.stuck[i] = stick_test(s, h, i) ? 1 : 0; s.removed[i] = 0; }
    else if (mode == SCAN_FINAL && s.removed[i]) s.stuck[i] = 0;
  }
  const int c = (i < s.N) ? scan_class(s, mode, i) : -1;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const unsigned mk = __ballot_sync(0xffffffffu, c == k);
    if ((threadIdx.x & 31) == 0 && mk) atomicAdd(&cnt[k], __popc(mk));
  }
  __syncthreads();
  if (threadIdx.x < 3) s.blk_cnt[threadIdx.x * nb + blockIdx.x] = cnt[threadIdx.x];
}

// single block: exclusive scan of the per-block counts, totals and cycle bookkeeping
__global__ void __launch_bounds__(256) k_scan_offsets(State s, int mode, int nb) {
  __shared__ int tot[3];
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (w < 3) {  // one warp per class, sequential over chunks of 32 blocks
    int run = 0;
    for (int b0 = 0; b0 < nb; b0 += 32) {
      const int b = b0 + lane;
      const int v = (b < nb) ? s.blk_cnt[w * nb + b] : 0;
      int inc = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int n = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += n; }
      if (b < nb) s.blk_cnt[w * nb + b] = run + inc - v;
      run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) tot[w] = run;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    Ctrl *c = s.ctrl;
    if (mode == SCAN_STICK || mode == SCAN_STICK_FLAGS) {
      c->nP0 = tot[1]; c->n_stuck = tot[1]; c->k_lost = 0; c->n_active = s.N - tot[1];
    } else if (mode == SCAN_FINAL) {
      c->nA = tot[0]; c->nP = tot[1]; c->nR = tot[2];
      c->k_lost = tot[2]; c->n_stuck = tot[1]; c->n_active = tot[0];
      c->strategy = 0;                                     // no reseeding yet in this cycle (and none on the last one)
      // Golden Rooster self-disable (R-9): two consecutive GR cycles without new peaks
      if (c->gr_used_last) {
        if (tot[1] > c->gr_prev_modes) c->gr_unproductive = 0; else c->gr_unproductive += 1;
        if (c->gr_unproductive >= 2) c->gr_enabled = 0;
      }
    } else {
      c->nE = tot[1];
      c->n_active = tot[1];                                // who takes part in phases 5-6 (= N - n_stuck after reseeding)
    }
  }
}

__global__ void __launch_bounds__(SCAN_BLOCK) k_scan_scatter(State s, int mode, int nb) {
  __shared__ int wcnt[3][SCAN_BLOCK / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int i = blockIdx.x * SCAN_BLOCK + threadIdx.x;
  const int c = (i < s.N) ? scan_class(s, mode, i) : -1;
  if (mode == SCAN_FINAL && i < s.N) { s.rs_src[i] = -1; s.rs_cand[i] = -1; }
  int rank = 0;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const unsigned mk = __ballot_sync(0xffffffffu, c == k);
    if (lane == 0) wcnt[k][w] = __popc(mk);
    if (c == k) rank = __popc(mk & ((1u << lane) - 1u));
  }
  __syncthreads();
  if (c >= 0) {
    int off = s.blk_cnt[c * nb + blockIdx.x] + rank;
    for (int ww = 0; ww < w; ++ww) off += wcnt[c][ww];
    int32_t *dst = (mode == SCAN_STICK || mode == SCAN_STICK_FLAGS) ? s.listP0 : (mode == SCAN_EXPLORE) ? s.listE
                   : (c == 0 ? s.listA : (c == 1 ? s.listP : s.listR));
    dst[off] = i;
  }
}

// The whole ordered scan in ONE launch for small populations (N <= SCAN_SMALL_MAX: C1, C2 -- launch-bound configurations,
// where the three kernels above cost three launch latencies for a few microseconds of work): one CTA walks the chunks of
// 1024 samples in order, keeps a running offset per class, and scatters at once; same flags, lists (ascending) and
// bookkeeping as k_scan_count + k_scan_offsets + k_scan_scatter.
static_assert(SCAN_SMALL_MAX % SCAN_BLOCK == 0, "whole chunks");
__global__ void __launch_bounds__(SCAN_BLOCK) k_scan_small(State s, Hyper h, int mode, int nb) {
  __shared__ int wcnt[3][SCAN_BLOCK / 32];
  __shared__ int run[3];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x < 3) run[threadIdx.x] = 0;
  __syncthreads();
  for (int b = 0; b < nb; ++b) {
    const int i = b * SCAN_BLOCK + threadIdx.x;
    if (i < s.N) {
      if (mode == SCAN_STICK_FLAGS) { s.stuck[i] = stick_test(s, h, i) ? 1 : 0; s.removed[i] = 0; }
      else if (mode == SCAN_FINAL && s.removed[i]) s.stuck[i] = 0;
      if (mode == SCAN_FINAL) { s.rs_src[i] = -1; s.rs_cand[i] = -1; }
    }
    const int c = (i < s.N) ? scan_class(s, mode, i) : -1;
    int rank = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const unsigned mk = __ballot_sync(0xffffffffu, c == k);
      if (lane == 0) wcnt[k][w] = __popc(mk);
      if (c == k) rank = __popc(mk & ((1u << lane) - 1u));
    }
    __syncthreads();
    if (c >= 0) {
      int off = run[c] + rank;
      for (int ww = 0; ww < w; ++ww) off += wcnt[c][ww];
      int32_t *dst = (mode == SCAN_STICK || mode == SCAN_STICK_FLAGS) ? s.listP0 : (mode == SCAN_EXPLORE) ? s.listE
                     : (c == 0 ? s.listA : (c == 1 ? s.listP : s.listR));
      dst[off] = i;
    }
    __syncthreads();
    if (threadIdx.x < 3) { int t = 0; for (int ww = 0; ww < SCAN_BLOCK / 32; ++ww) t += wcnt[threadIdx.x][ww]; run[threadIdx.x] += t; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    Ctrl *c = s.ctrl;
    const int tot[3] = {run[0], run[1], run[2]};
    if (mode == SCAN_STICK || mode == SCAN_STICK_FLAGS) {
      c->nP0 = tot[1]; c->n_stuck = tot[1]; c->k_lost = 0; c->n_active = s.N - tot[1];
    } else if (mode == SCAN_FINAL) {
      c->nA = tot[0]; c->nP = tot[1]; c->nR = tot[2];
      c->k_lost = tot[2]; c->n_stuck = tot[1]; c->n_active = tot[0];
      c->strategy = 0;
      if (c->gr_used_last) {                                  // Golden Rooster self-disable (R-9)
        if (tot[1] > c->gr_prev_modes) c->gr_unproductive = 0; else c->gr_unproductive += 1;
        if (c->gr_unproductive >= 2) c->gr_enabled = 0;
      }
    } else {
      c->nE = tot[1];
      c->n_active = tot[1];
    }
  }
}

static cudaError_t run_scan(const State &s, const Hyper &h, int mode, cudaStream_t st) {
  const int nb = (s.N + SCAN_BLOCK - 1) / SCAN_BLOCK;
  if (nb == 0) {  // empty population: only the bookkeeping kernel runs
    k_scan_offsets<<<1, 256, 0, st>>>(s, mode, 0);
    return cudaGetLastError();
  }
  if (s.N <= SCAN_SMALL_MAX) {
    k_scan_small<<<1, SCAN_BLOCK, 0, st>>>(s, h, mode, nb);
    return cudaGetLastError();
  }
  k_scan_count<<<nb, SCAN_BLOCK, 0, st>>>(s, h, mode, nb);
  k_scan_offsets<<<1, 256, 0, st>>>(s, mode, nb);
  k_scan_scatter<<<nb, SCAN_BLOCK, 0, st>>>(s, mode, nb);
  return cudaGetLastError();
}

// ---- Phase 3 (Eq. 4; R-7): removed_i = stuck_i and exists j != i stuck within eps_dup in
// L-infinity with f_j > f_i or (f_j = f_i and j < i); every test against the pre-removal stuck set. ------
// Thread = one stuck sample i (its row in registers); a CTA of 128 samples walks ONE of DEDUP_SPLIT slices of the stuck list
// in 64-row shared-memory tiles (rows as float4, read by all threads at once: broadcast).  Per pair: the f / index rule
// first (it discards half of the pairs), then coordinate 0 (it discards almost every pair of different clusters), then
// the remaining coordinates eight at a time with an early exit.  The slices of a sample's comparison run in different CTAs
// (grid.y), so that a few hundred blocks of stuck samples still fill 148 SMs; a slice that finds a dominating
// duplicate sets removed[i] (the mask is zero before the launch).  Worst case measured at C5 -- 52 % of N = 65536 stuck in
// 300 clusters, 1.2e9 pairs -- in profiles/r2_worstcase_select_c5.md.
constexpr int DEDUP_TILE = 64;
constexpr int DEDUP_SPLIT = 8;
__global__ void __launch_bounds__(128) k_dedup(State s, Hyper h) {
  __shared__ float4 tx[DEDUP_TILE][CHISAO_MAX_D / 4];
  __shared__ float tf[DEDUP_TILE];
  __shared__ int ti[DEDUP_TILE];
  const int n = s.ctrl->nP0, d = s.d;
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (blockIdx.x * blockDim.x >= n) return;
  const int per = (((n + DEDUP_SPLIT - 1) / DEDUP_SPLIT) + DEDUP_TILE - 1) / DEDUP_TILE * DEDUP_TILE;   // slice length, whole tiles
  const int jbeg = blockIdx.y * per, jend = min(n, jbeg + per);
  if (jbeg >= n) return;
  const bool act = q < n;
  const int i = act ? s.listP0[q] : -1;
  float xi[CHISAO_MAX_D];
#pragma unroll
  for (int c = 0; c < CHISAO_MAX_D; ++c) xi[c] = (act && c < d) ? s.x[(size_t)i * d + c] : 0.0f;
  const float fi = act ? s.f[i] : 0.0f;
  const float eps = h.eps_dup;
  const int d4 = (d + 3) / 4;
  bool rem = false;
  for (int j0 = jbeg; j0 < jend; j0 += DEDUP_TILE) {
    __syncthreads();
    for (int e = threadIdx.x; e < DEDUP_TILE * d4; e += blockDim.x) {
      const int r = e / d4, c4 = e - r * d4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (j0 + r < jend) {
        const float *row = s.x + (size_t)s.listP0[j0 + r] * d;
        v.x = row[4 * c4];
        if (4 * c4 + 1 < d) v.y = row[4 * c4 + 1];
        if (4 * c4 + 2 < d) v.z = row[4 * c4 + 2];
        if (4 * c4 + 3 < d) v.w = row[4 * c4 + 3];
      }
      tx[r][c4] = v;
    }
    if (threadIdx.x < DEDUP_TILE) {
      const int jj = j0 + threadIdx.x;
      ti[threadIdx.x] = (jj < jend) ? s.listP0[jj] : -1;
      tf[threadIdx.x] = (jj < jend) ? s.f[s.listP0[jj]] : 0.0f;
    }
    __syncthreads();
    if (act && !rem) {
      const int lim = min(DEDUP_TILE, jend - j0);
      for (int r = 0; r < lim && !rem; ++r) {
        const int j = ti[r];
        const float fj = tf[r];
        if (j == i || !(fj > fi || (fj == fi && j < i))) continue;   // Eq. 4 (R-7): only a better (or equal and earlier) sample removes i
        if (!(fabsf(xi[0] - tx[r][0].x) < eps)) continue;
        bool close = true;
#pragma unroll
        for (int c4 = 0; c4 < CHISAO_MAX_D / 4; ++c4) {
          if (4 * c4 < d) {
            const float4 v = tx[r][c4];                      // (coordinates beyond d are zero on both sides)
            close = close && (fabsf(xi[4 * c4] - v.x) < eps) && (fabsf(xi[4 * c4 + 1] - v.y) < eps) &&
                    (fabsf(xi[4 * c4 + 2] - v.z) < eps) && (fabsf(xi[4 * c4 + 3] - v.w) < eps);
          }
          if ((c4 & 1) == 1 && !close) break;
        }
        rem = close;
      }
    }
  }
  if (act && rem) s.removed[i] = 1;
}

// have_partials: ||grad f||_inf per sample and f_max were written by the last L-BFGS update of the pass
// (k_lbfgs_update<STICK>, chisao_lbfgs.cu); otherwise (stand-alone unit, n_conv = 0) k_ginf_fmax computes them here
cudaError_t launch_stick(const State &s, const Hyper &h, bool have_partials, cudaStream_t st) {
  if (!have_partials) {
    cudaError_t e = cudaMemsetAsync(&s.ctrl->fmax_enc, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    if (s.N > 0) k_ginf_fmax<<<(s.N + 7) / 8, 256, 0, st>>>(s);
  }
  return run_scan(s, h, SCAN_STICK_FLAGS, st);
}

cudaError_t launch_dedup(const State &s, const Hyper &h, bool rebuild_p0, cudaStream_t st) {
  if (s.N > 0) {
    // as a stand-alone unit (chisao_phase) the caller may have edited the flags: rebuild the pre-removal stuck list
    // first; inside a cycle launch_stick has just written it
    cudaError_t e = cudaSuccess;
    if (rebuild_p0) {
      e = run_scan(s, h, SCAN_STICK, st);
      if (e != cudaSuccess) return e;
      e = cudaMemsetAsync(s.removed, 0, s.N, st);          // (inside a cycle the stick test has just cleared the mask)
      if (e != cudaSuccess) return e;
    }
    if (h.phase_mask & (1u << 3)) k_dedup<<<dim3((s.N + 127) / 128, DEDUP_SPLIT), 128, 0, st>>>(s, h);
  }
  return run_scan(s, h, SCAN_FINAL, st);                   // its counting kernel clears the stuck flag of removed samples
}

cudaError_t launch_explore_list(const State &s, cudaStream_t st) { Hyper h{}; return run_scan(s, h, SCAN_EXPLORE, st); }

// ---- Phase 4: reseeding ---------------------------------------------------------------
// strategy decision + Golden-Rooster basis: QR of a Gaussian d x d matrix by modified Gram-Schmidt with one
// re-orthogonalisation pass, R_ii > 0 (R-9).  Single CTA.
__global__ void __launch_bounds__(256) k_reseed_prepare(State s, Hyper h, int cycle) {
  __shared__ float Q[CHISAO_MAX_D][CHISAO_MAX_D + 1];   // Q[r][c]
  __shared__ int strat;
  const int d = s.d, t = threadIdx.x, lane = t & 31, w = t >> 5;
  if (t == 0) {
    Ctrl *c = s.ctrl;
    int st = 0;
    c->gr_used_last = 0;
    if (c->k_lost > 0 && (h.phase_mask & (1u << 4))) {
      if (c->nA >= 5) st = 1;                                // Repulse Monkey
      else if (c->gr_enabled && c->nP > 0) { st = 2; c->gr_used_last = 1; c->gr_prev_modes = c->nP; }
      else st = 3;                                           // population kept at N (R-9)
    }
    c->strategy = st;
    strat = st;
  }
  __syncthreads();
  if (strat != 2) return;
  for (int e = t; e < d * d; e += blockDim.x)
    Q[e / d][e % d] = rng_normal(h.seed, 0u, (uint32_t)cycle, rng_tag(4, 0, PUR_GR_MATRIX), (uint32_t)e);
  __syncthreads();
  if (w == 0) {  // modified Gram-Schmidt, twice per column, by one warp (lane L owns rows L and L + 32)
    for (int c = 0; c < d; ++c) {
      for (int pass = 0; pass < 2; ++pass) {
        for (int e = 0; e < c; ++e) {
          float part = 0.0f;
          for (int r = lane; r < d; r += 32) part = fmaf(Q[r][e], Q[r][c], part);
          const float dot = warp_sum(part);
          for (int r = lane; r < d; r += 32) Q[r][c] = fmaf(-dot, Q[r][e], Q[r][c]);
          __syncwarp();
        }
      }
      float part = 0.0f;
      for (int r = lane; r < d; r += 32) part = fmaf(Q[r][c], Q[r][c], part);
      const float inv = 1.0f / sqrtf(warp_sum(part));
      for (int r = lane; r < d; r += 32) Q[r][c] *= inv;
      __syncwarp();
    }
  }
  __syncthreads();
  for (int e = t; e < d * d; e += blockDim.x) s.grQ[e] = Q[e / d][e % d];
}

// distance along direction u from x to the boundary of Theta (one-sided ray); warp-cooperative
__device__ __forceinline__ float ray_exit(float xa, float xb, float ua, float ub, float loa, float lob, float hia,
                                          float hib, bool va, bool vb) {
  float ta = INFINITY, tb = INFINITY;
  if (va) { if (ua > 0.f) ta = (hia - xa) / ua; else if (ua < 0.f) ta = (loa - xa) / ua; }
  if (vb) { if (ub > 0.f) tb = (hib - xb) / ub; else if (ub < 0.f) tb = (lob - xb) / ub; }
  float tm = warp_min(fminf(ta, tb));
  if (!(tm >= 0.0f) || !(tm <= 3.0e38f)) tm = 0.0f;
  return tm;
}

constexpr int RS_WARPS = 4;
constexpr int RS_MAXC = 16;
// one warp per removed slot q (rank in the ascending list R); lane L owns coordinates L and L + 32
__global__ void __launch_bounds__(RS_WARPS * 32) k_reseed(State s, Hyper h, int cycle) {
  __shared__ float cand[RS_WARPS][RS_MAXC][CHISAO_MAX_D];
  const Ctrl *c = s.ctrl;
  const int strat = c->strategy;
  if (strat == 0) return;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int q = blockIdx.x * RS_WARPS + w;
  const int nR = c->nR, nA = c->nA, nP = c->nP, d = s.d;
  if (q >= nR) return;
  const int r = s.listR[q];
  const int ja = lane, jb = lane + 32;
  const bool va = ja < d, vb = jb < d;
  const float loa = va ? s.lo[ja] : 0.f, hia = va ? s.hi[ja] : 0.f;
  const float lob = vb ? s.lo[jb] : 0.f, hib = vb ? s.hi[jb] : 0.f;
  float outa = 0.f, outb = 0.f;
  int src = -1, chosen = -1;
  if (strat == 1) {
    // Repulse Monkey (R-8): ray from a random unfrozen sample in a random direction, C uniform
    // candidates along it inside Theta, keep the one farthest (min L2) from the frozen-mode set P
    const uint4 w0 = philox_block(h.seed, 0u, (uint32_t)r, (uint32_t)cycle, rng_tag(4, 0, PUR_RS_SRC));
    src = s.listA[(int)(((unsigned long long)w0.x * (unsigned long long)nA) >> 32)];
    const uint32_t tdir = rng_tag(4, 0, PUR_RS_DIR), tt = rng_tag(4, 0, PUR_RS_T);
    float ua = va ? rng_normal(h.seed, (uint32_t)r, (uint32_t)cycle, tdir, (uint32_t)ja) : 0.f;
    float ub = vb ? rng_normal(h.seed, (uint32_t)r, (uint32_t)cycle, tdir, (uint32_t)jb) : 0.f;
    const float nrm = sqrtf(warp_sum(fmaf(ua, ua, ub * ub)));
    ua /= nrm; ub /= nrm;
    const float xa = va ? s.x[(size_t)src * d + ja] : 0.f, xb = vb ? s.x[(size_t)src * d + jb] : 0.f;
    const float tmax = ray_exit(xa, xb, ua, ub, loa, lob, hia, hib, va, vb);
    const int C = h.reseed_cands;
    for (int cc = 0; cc < C; ++cc) {
      const float U = rng_uniform(h.seed, (uint32_t)r, (uint32_t)cycle, tt, (uint32_t)cc);
      if (va) cand[w][cc][ja] = clipf(fmaf(tmax * U, ua, xa), loa, hia);
      if (vb) cand[w][cc][jb] = clipf(fmaf(tmax * U, ub, xb), lob, hib);
    }
    __syncwarp();
    float mind[RS_MAXC];
#pragma unroll
    for (int cc = 0; cc < RS_MAXC; ++cc) mind[cc] = INFINITY;
    for (int pi = lane; pi < nP; pi += 32) {
      const float *xp = s.x + (size_t)s.listP[pi] * d;
      float d2[RS_MAXC];
#pragma unroll
      for (int cc = 0; cc < RS_MAXC; ++cc) d2[cc] = 0.f;
      for (int j = 0; j < d; ++j) {
        const float xv = xp[j];
#pragma unroll
        for (int cc = 0; cc < RS_MAXC; ++cc)
          if (cc < C) { const float e = cand[w][cc][j] - xv; d2[cc] = fmaf(e, e, d2[cc]); }
      }
#pragma unroll
      for (int cc = 0; cc < RS_MAXC; ++cc) if (cc < C) mind[cc] = fminf(mind[cc], d2[cc]);
    }
    float best = -1.0f;
    chosen = 0;
#pragma unroll
    for (int cc = 0; cc < RS_MAXC; ++cc) {
      if (cc < C) {
        const float mm = warp_min(mind[cc]);
        if (mm > best) { best = mm; chosen = cc; }
      }
    }
    if (va) outa = cand[w][chosen][ja];
    if (vb) outb = cand[w][chosen][jb];
  } else if (strat == 2) {
    // Golden Rooster (R-9): ray from a confirmed peak along +/- an orthonormal direction
    const int peak = s.listP[q % nP], col = (q / nP) % d;
    const int neg = (int)(((long long)q / ((long long)nP * d)) % 2);
    float ua = va ? s.grQ[ja * d + col] : 0.f, ub = vb ? s.grQ[jb * d + col] : 0.f;
    if (neg) { ua = -ua; ub = -ub; }
    const float xa = va ? s.x[(size_t)peak * d + ja] : 0.f, xb = vb ? s.x[(size_t)peak * d + jb] : 0.f;
    const float tmax = ray_exit(xa, xb, ua, ub, loa, lob, hia, hib, va, vb);
    const float U = rng_uniform(h.seed, (uint32_t)r, (uint32_t)cycle, rng_tag(4, 0, PUR_RS_T), 0u);
    outa = clipf(fmaf(tmax * U, ua, xa), loa, hia);
    outb = clipf(fmaf(tmax * U, ub, xb), lob, hib);
    src = peak; chosen = col * 2 + neg;
  } else {
    const uint32_t tu = rng_tag(4, 0, PUR_RS_UNIF);
    if (va) outa = clipf(fmaf(rng_uniform(h.seed, (uint32_t)r, (uint32_t)cycle, tu, (uint32_t)ja), hia - loa, loa), loa, hia);
    if (vb) outb = clipf(fmaf(rng_uniform(h.seed, (uint32_t)r, (uint32_t)cycle, tu, (uint32_t)jb), hib - lob, lob), lob, hib);
  }
  // "All reseeded samples are marked as unstuck"; velocity and history reset
  if (va) { s.x[(size_t)r * d + ja] = outa; s.v[(size_t)r * d + ja] = 0.f; }
  if (vb) { s.x[(size_t)r * d + jb] = outb; s.v[(size_t)r * d + jb] = 0.f; }
  if (lane == 0) {
    s.removed[r] = 0; s.stuck[r] = 0; s.hist_len[r] = 0; s.hist_head[r] = 0;
    s.rs_src[r] = src; s.rs_cand[r] = chosen;
  }
}

__global__ void k_reseed_finish(State s) {
  Ctrl *c = s.ctrl;
  if (c->strategy != 0) c->n_active = s.N - c->n_stuck;
}

// standalone (chisao_phase): reset the diagnostics and fix n_active here; inside a cycle the list kernels before and
// after this phase do both (k_scan_scatter SCAN_FINAL, k_scan_offsets SCAN_EXPLORE)
cudaError_t launch_reseed(const State &s, const Hyper &h, int cycle, bool standalone, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  if (standalone) {
    cudaError_t e = cudaMemsetAsync(s.rs_src, 0xFF, sizeof(int32_t) * s.N, st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(s.rs_cand, 0xFF, sizeof(int32_t) * s.N, st);
    if (e != cudaSuccess) return e;
  }
  k_reseed_prepare<<<1, 256, 0, st>>>(s, h, cycle);
  k_reseed<<<(s.N + RS_WARPS - 1) / RS_WARPS, RS_WARPS * 32, 0, st>>>(s, h, cycle);
  if (standalone) k_reseed_finish<<<1, 1, 0, st>>>(s);
  return cudaGetLastError();
}

// ---- smoothing scale of Hands Like Clouds (R-18): sigma_s > 0 as given, else c * pooled population
// std over all coordinates of the unfrozen samples (c = |sigma_s|), re-estimated at every step -------------------
__global__ void __launch_bounds__(256) k_sigma_sum(State s) {
  __shared__ double shx[8], shxx[8];
  const int nE = s.ctrl->nE, d = s.d;
  const size_t n = (size_t)nE * d;
  double a = 0.0, b = 0.0;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
    const int q = (int)(e / d), j = (int)(e - (size_t)q * d);
    const double v = (double)s.x[(size_t)s.listE[q] * d + j];
    a += v; b += v * v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
  if ((threadIdx.x & 31) == 0) { shx[threadIdx.x >> 5] = a; shxx[threadIdx.x >> 5] = b; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) { a += shx[w]; b += shxx[w]; }
    atomicAdd(&s.ctrl->sx, a); atomicAdd(&s.ctrl->sxx, b);
  }
}
__global__ void k_sigma_final(State s, Hyper h) {
  Ctrl *c = s.ctrl;
  if (h.sigma_s > 0.0f) { c->sigma_eff = h.sigma_s; return; }
  const double n = (double)c->nE * (double)s.d;
  if (n == 0.0) { c->sigma_eff = 0.0f; return; }
  const double mean = c->sx / n, var = fmax(c->sxx / n - mean * mean, 0.0);
  c->sigma_eff = (float)(fabs((double)h.sigma_s) * sqrt(var));
}
// a caller-supplied scale (sigma_s > 0) is written to ctrl->sigma_eff once, at chisao_init: nothing to launch then
cudaError_t launch_hlc_sigma(const State &s, const Hyper &h, cudaStream_t st) {
  if (h.sigma_s > 0.0f) return cudaSuccess;
  if (s.N > 0) {
    cudaError_t e = cudaMemsetAsync(&s.ctrl->sx, 0, 2 * sizeof(double), st);
    if (e != cudaSuccess) return e;
    k_sigma_sum<<<148, 256, 0, st>>>(s);
  }
  k_sigma_final<<<1, 1, 0, st>>>(s, h);
  return cudaGetLastError();
}

// ---- Hands Like Clouds, the paper's own form, Eq. 5 (DESIGN.md NEXT-2) -----------------------
// theta <- theta + eta (1/K) sum_k grad f(theta + sigma z_k) with FD gradients: per draw k the host runs
// [perturb: xt = x + sigma z_k] -> k_eval_fd on xt (noise slots k 2d + ..) -> [accumulate: ghat += gn / K], then
// [apply].  One thread per (explore-list entry, coordinate).
__global__ void k_hlc5(State s, Hyper h, int cycle, int iter, int k, int stage) {
  const int nE = s.ctrl->nE, d = s.d;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (size_t)nE * d || s.ctrl->sigma_eff == 0.0f) return;   // sigma = 0: nobody moves (R-18)
  const int q = (int)(e / d), j = (int)(e - (size_t)q * d);
  const int i = s.listE[q];
  const size_t o = (size_t)i * d + j;
  if (stage == 0) {
    const float u = rng_normal(h.seed, (uint32_t)i, (uint32_t)cycle, rng_tag(5, iter, PUR_HLC_U), (uint32_t)(k * d + j));
    s.xt[o] = fmaf(s.ctrl->sigma_eff, u, s.x[o]);         // evaluation points are not clipped (R-12)
  } else if (stage == 1) {
    s.ghat[o] = (k == 0 ? 0.0f : s.ghat[o]) + s.gn[o] / (float)h.hlc_M;
  } else {
    s.x[o] = clipf(fmaf(h.eta_hlc, s.ghat[o], s.x[o]), s.lo[j], s.hi[j]);
  }
}
cudaError_t launch_hlc5(const State &s, const Hyper &h, int cycle, int iter, int k, int stage, cudaStream_t st) {
  const size_t n = (size_t)s.N * s.d;
  if (n == 0) return cudaSuccess;
  k_hlc5<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(s, h, cycle, iter, k, stage);
  return cudaGetLastError();
}

// ---- initial population: i.i.d. uniform in Theta (Prop. 2; R-15 purpose INIT, cycle 0) -------
__global__ void k_seed_population(State s, Hyper h) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (size_t)s.N * s.d) return;
  const int i = (int)(e / s.d), j = (int)(e % s.d);
  const float U = rng_uniform(h.seed, (uint32_t)i, 0u, rng_tag(0, 0, PUR_INIT), (uint32_t)j);
  s.x[e] = clipf(fmaf(U, s.hi[j] - s.lo[j], s.lo[j]), s.lo[j], s.hi[j]);
}
cudaError_t launch_seed_population(const State &s, const Hyper &h, cudaStream_t st) {
  const size_t n = (size_t)s.N * s.d;
  if (n == 0) return cudaSuccess;
  k_seed_population<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(s, h);
  return cudaGetLastError();
}

__global__ void k_gather_rows(const float *x, const int32_t *idx, int n, int d, float *out) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (size_t)n * d) return;
  const int q = (int)(e / d), j = (int)(e % d);
  out[e] = x[(size_t)idx[q] * d + j];
}
cudaError_t launch_gather_rows(const float *x, const int32_t *idx, int n, int d, float *out, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  k_gather_rows<<<(unsigned)(((size_t)n * d + 255) / 256), 256, 0, st>>>(x, idx, n, d, out);
  return cudaGetLastError();
}

}  // namespace chisao
