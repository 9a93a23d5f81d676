// chisao_eval_kernels.cuh -- the three evaluation kernels (see chisao_eval.cuh) and their launchers,
// instantiated once per objective id in chisao_eval_obj.cu (-DCHISAO_OBJ_INST=<id>).
#pragma once
#include "chisao_eval.cuh"

namespace chisao {

// all lanes of the warp must call; returns the slot for lanes with pred, -1 otherwise
__device__ __forceinline__ int warp_append(int32_t *counter, bool pred) {
  const unsigned mask = __ballot_sync(0xffffffffu, pred);
  if (mask == 0u) return -1;
  const int lane = threadIdx.x & 31, leader = __ffs(mask) - 1;
  int base = 0;
  if (lane == leader) base = atomicAdd(counter, __popc(mask));
  base = __shfl_sync(0xffffffffu, base, leader);
  return pred ? base + __popc(mask & ((1u << lane) - 1u)) : -1;
}

struct FdArgs {
  const float *X;            // [N][d] points the stencil is centred on (x or xt)
  const int32_t *list;       // sample ids (NULL = identity)
  const int32_t *count;      // device count (NULL = max_count)
  int32_t max_count, mode, d, cycle, phase, iter, counter;
  int32_t slot_off;          // added to the noise slot (paper-form HLC: draw k uses slots k 2d + 1 ..)
  float *g_out;              // FD_GRAD: [N][d]
  float *x, *v;              // FD_ANTI: updated in place
  const float *lo, *hi;
  float h, mu, alpha;
  uint64_t seed;
  unsigned long long *evals;
  int32_t *zero_cnt;         // counter reset by the kernel (the consumed line-search worklist), or NULL
};

// stencil-aware FD evaluator for the dense objectives (chisao_stencil.cu; opt-in)
bool fd_stencil_supported(const DevObj &o);
cudaError_t launch_fd_stencil(const DevObj &o, const FdArgs &a, int n_samples, cudaStream_t st);

// ---- central finite differences: 2d stencil points per sample (R-1) ---------------
// thread t -> (sample t / d of the tile, coordinate j = t % d); it evaluates both x + h e_j and x - h e_j
// (noise slots 1 + 2j and 2 + 2j, R-2) and forms g_j with the step actually taken in fp32.
template <int OBJ, int DP>
__global__ void __launch_bounds__(NT, 2) k_eval_fd(const DevObj o, const FdArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const EvalSmem sm = carve_smem<DP>(smem_raw, o.kc * o.rec);
  const int t = threadIdx.x, d = a.d;
  const int spt = NT / d;                          // samples per tile
  const int cnt = a.count ? *a.count : a.max_count;
  const int first = blockIdx.x * spt;
  if (blockIdx.x == 0 && t == 0 && a.zero_cnt) *a.zero_cnt = 0;
  if (first >= cnt) return;
  if (t == 0) { mbar_init(&sm.bar[0], 1); mbar_init(&sm.bar[1], 1); mbar_fence_init(); }
  const int s = t / d, j = t - s * d;
  const bool valid = (s < spt) && (first + s < cnt);
  const int i = valid ? (a.list ? a.list[first + s] : first + s) : 0;
  const bool vec = (d & 3) == 0;
  float xj = 0.f, xph = 0.f, xmh = 0.f;
  if (valid) {
    const float *row = a.X + (size_t)i * d;
    xj = row[j]; xph = xj + a.h; xmh = xj - a.h;
#pragma unroll
    for (int c4 = 0; c4 < DP / 4; ++c4) {
      const float4 v = ld_row4(row, c4, d, vec);
      float4 vp = v, vm = v;
      if (c4 == (j >> 2)) { set4(vp, j & 3, xph); set4(vm, j & 3, xmh); }
      sm.pts[c4 * PTILE + t] = vp;
      sm.pts[c4 * PTILE + NT + t] = vm;
    }
  } else {
#pragma unroll
    for (int c4 = 0; c4 < DP / 4; ++c4) {
      sm.pts[c4 * PTILE + t] = make_float4(0.f, 0.f, 0.f, 0.f);
      sm.pts[c4 * PTILE + NT + t] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  __syncthreads();
  uint32_t use = 0;
  float fv[PPT];
  eval_tile<OBJ, DP>(o, sm, t, use, fv);
  if (valid) {
    const float fp = fv[0] + eval_noise(o.sigma_noise, a.seed, a.cycle, i, a.phase, a.iter, a.slot_off + 1 + 2 * j);
    const float fm = fv[1] + eval_noise(o.sigma_noise, a.seed, a.cycle, i, a.phase, a.iter, a.slot_off + 2 + 2 * j);
    const float g = (fp - fm) / ((xph - xj) + (xj - xmh));
    if (a.mode == FD_GRAD) {
      a.g_out[(size_t)i * d + j] = g;
    } else {  // Eq. 6: v <- mu v - alpha grad f;  x <- x + v, clipped to Theta (R-12)
      const float vo = (a.iter == 1) ? 0.0f : a.v[(size_t)i * d + j];
      const float vn = fmaf(a.mu, vo, -a.alpha * g);
      a.v[(size_t)i * d + j] = vn;
      a.x[(size_t)i * d + j] = clipf(xj + vn, a.lo[j], a.hi[j]);
    }
  }
  if (t == 0) atomicAdd(&a.evals[a.counter], (unsigned long long)min(spt, cnt - first) * 2ull * d);
}

struct PtArgs {
  const float *X;            // centre: x; line search: xt
  const int32_t *list;
  const int32_t *count;
  int32_t max_count, mode, b, d, cycle, iter, ls_max;
  float *f;                  // [N] current values
  float *ft, *dec, *tcur;    // [N] trial value, Armijo linear term, current step
  float *xt;                 // [N][d] trial points (rewritten on reject)
  const float *x, *p, *g, *lo, *hi;
  int32_t *ls_b, *next_list, *next_cnt, *fd_list, *fd_cnt, *zero_cnt;
  int32_t rows_in_smem;      // PT_LS_ALL: the launch carries 3 x [DP/4][PTILE] float4 of extra shared memory for the rows x, p, g
  int32_t tc_pts;            // PT_LS_ALL on the tensor-core evaluators: worklist entries per CTA, 256 or 128 (set by launch_pt_tc)
  float c1, shrink;
  uint64_t seed;
  unsigned long long *evals;
};

// Line-search retry (R-4): the shrunk trial point x_t = clip(x + t p) of sample i and the directional decrease
// -g . (x_t - x), accumulated in coordinate order.  Rows are fetched eight coordinates at a time (independent loads in
// flight) before anything is stored: a scalar loop serialises on the L2 latency of every coordinate.
__device__ __forceinline__ float ls_retry_row(const PtArgs &a, int i, int d, float tn) {
  const float *__restrict__ xr = a.x + (size_t)i * d;
  const float *__restrict__ pr = a.p + (size_t)i * d;
  const float *__restrict__ gr = a.g + (size_t)i * d;
  float *xt = a.xt + (size_t)i * d;
  float dsum = 0.0f;
  int j = 0;
  if ((d & 3) == 0) {
    for (; j + 8 <= d; j += 8) {
      const float4 x0 = *reinterpret_cast<const float4 *>(xr + j), x1 = *reinterpret_cast<const float4 *>(xr + j + 4);
      const float4 p0 = *reinterpret_cast<const float4 *>(pr + j), p1 = *reinterpret_cast<const float4 *>(pr + j + 4);
      const float4 g0 = *reinterpret_cast<const float4 *>(gr + j), g1 = *reinterpret_cast<const float4 *>(gr + j + 4);
      const float xo[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
      const float pv[8] = {p0.x, p0.y, p0.z, p0.w, p1.x, p1.y, p1.z, p1.w};
      const float gv[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
      float xn[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        xn[e] = clipf(fmaf(tn, pv[e], xo[e]), a.lo[j + e], a.hi[j + e]);
        dsum = fmaf(-gv[e], xn[e] - xo[e], dsum);
      }
      *reinterpret_cast<float4 *>(xt + j) = make_float4(xn[0], xn[1], xn[2], xn[3]);
      *reinterpret_cast<float4 *>(xt + j + 4) = make_float4(xn[4], xn[5], xn[6], xn[7]);
    }
  }
  for (; j < d; ++j) {
    const float xo = xr[j];
    const float xn = clipf(fmaf(tn, pr[j], xo), a.lo[j], a.hi[j]);
    xt[j] = xn;
    dsum = fmaf(-gr[j], xn - xo, dsum);
  }
  return dsum;
}

// the Armijo decision of one line-search trial (R-4 (iv)); a non-finite trial value is rejected (R-12)
__device__ __forceinline__ bool ls_accept(float val, float f_i, float dec_i, float c1) {
  const float phit = -val, phi = -f_i;
  const float rhs = fmaf(c1, dec_i, phi);                 // Armijo: phi_t <= phi + c1 gamma.(x_t - x)
  return (fabsf(phit) <= 3.0e38f) && (phit <= rhs);
}

// ---- one point per sample: cycle-start centre value, or line-search trial b (R-4) ---------------------
// PT_LS     : trial b of the samples on worklist b % 3; rejected samples are compacted onto worklist (b + 1) % 3
//             (one launch per trial: for evaluators whose tile is expensive, the retries stay dense)
// PT_LS_ALL : every trial b = 0 .. ls_max of the samples on worklist 0 in ONE launch: a tile keeps its samples and
//             repeats evaluate -> Armijo -> shrink until none of them retries (for evaluators whose tile costs
//             microseconds: the ls_max + 1 dependent launches, most of them empty, were the cost)
// Both forms run the same per-sample arithmetic (same evaluator, noise slot 2d + 1 + b, Armijo test, shrink).
template <int OBJ, int DP>
__global__ void __launch_bounds__(NT, 2) k_eval_points(const DevObj o, const PtArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const EvalSmem sm = carve_smem<DP>(smem_raw, o.kc * o.rec);
  const int t = threadIdx.x, d = a.d;
  const int cnt = a.count ? *a.count : a.max_count;
  const int first = blockIdx.x * PTILE;
  if (blockIdx.x == 0 && t == 0 && a.zero_cnt) *a.zero_cnt = 0;
  if (first >= cnt) return;
  if (t == 0) { mbar_init(&sm.bar[0], 1); mbar_init(&sm.bar[1], 1); mbar_fence_init(); }
  const bool vec = (d & 3) == 0;
  int idx[PPT]; bool valid[PPT];
  // PT_LS_ALL with rows_in_smem: the rows x, p, g of the thread's samples stay in shared memory for all rounds
  // (thread-private float4 columns like the staged points), f, the Armijo term and the step in registers: a round
  // touches global memory only for the bounds and, when a sample leaves the loop, for its results
  float4 *XS = reinterpret_cast<float4 *>(sm.extra), *PS = XS + (DP / 4) * PTILE, *GS = PS + (DP / 4) * PTILE;
  const bool rows = a.mode == PT_LS_ALL && a.rows_in_smem;
  float f_i[PPT], dec_i[PPT], t_i[PPT];
#pragma unroll
  for (int pp = 0; pp < PPT; ++pp) {
    const int e = first + pp * NT + t;
    valid[pp] = e < cnt;
    idx[pp] = valid[pp] ? (a.list ? a.list[e] : e) : 0;
    f_i[pp] = 0.f; dec_i[pp] = 0.f; t_i[pp] = 0.f;
    if (rows && valid[pp]) {
      const int i = idx[pp];
      f_i[pp] = a.f[i]; dec_i[pp] = a.dec[i]; t_i[pp] = a.tcur[i];
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        XS[c4 * PTILE + pp * NT + t] = ld_row4(a.x + (size_t)i * d, c4, d, vec);
        PS[c4 * PTILE + pp * NT + t] = ld_row4(a.p + (size_t)i * d, c4, d, vec);
        GS[c4 * PTILE + pp * NT + t] = ld_row4(a.g + (size_t)i * d, c4, d, vec);
      }
    }
  }
  uint32_t use = 0;
  unsigned int nev = 0;                                   // evaluations done by this thread (PT_LS_ALL)
  for (int b = a.b;; ++b) {
    if (!(rows && b > a.b)) {                             // (with the rows in shared memory, a retry has written its next point already)
#pragma unroll
      for (int pp = 0; pp < PPT; ++pp) {
        const float *row = a.X + (size_t)idx[pp] * d;
#pragma unroll
        for (int c4 = 0; c4 < DP / 4; ++c4)
          sm.pts[c4 * PTILE + pp * NT + t] = valid[pp] ? ld_row4(row, c4, d, vec) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
    __syncthreads();
    float fv[PPT];
    eval_tile<OBJ, DP>(o, sm, t, use, fv);
    bool again = false;
#pragma unroll
    for (int pp = 0; pp < PPT; ++pp) {
      const int i = idx[pp];
      bool accept = false, retry = false;
      float val = 0.f;
      if (valid[pp]) {
        if (a.mode == PT_CENTRE) {
          a.f[i] = fv[pp] + eval_noise(o.sigma_noise, a.seed, a.cycle, i, 1, 0, 0);
        } else {
          val = fv[pp] + eval_noise(o.sigma_noise, a.seed, a.cycle, i, 1, a.iter, 2 * d + 1 + b);
          accept = ls_accept(val, rows ? f_i[pp] : a.f[i], rows ? dec_i[pp] : a.dec[i], a.c1);
          retry = !accept && (b < a.ls_max);
          nev += 1u;
        }
      }
      if (a.mode != PT_CENTRE) {
        const int sa = warp_append(a.fd_cnt, accept);
        if (accept) { a.fd_list[sa] = i; a.ls_b[i] = b; a.ft[i] = val; }
        if (a.mode == PT_LS) {
          const int sr = warp_append(a.next_cnt, retry);
          if (retry) a.next_list[sr] = i;
        }
        if (rows) {
          const int col = pp * NT + t;
          if (valid[pp] && !retry && b > a.b) {           // the sample leaves the loop: its last trial point and step go back to the state
            a.tcur[i] = t_i[pp]; a.dec[i] = dec_i[pp];
            for (int c4 = 0; 4 * c4 < d; ++c4) {
              const float4 v = sm.pts[c4 * PTILE + col];
              float *dst = a.xt + (size_t)i * d + 4 * c4;
              if (vec) *reinterpret_cast<float4 *>(dst) = v;
              else {
                dst[0] = v.x;
                if (4 * c4 + 1 < d) dst[1] = v.y;
                if (4 * c4 + 2 < d) dst[2] = v.z;
                if (4 * c4 + 3 < d) dst[3] = v.w;
              }
            }
          }
          if (retry) {   // same arithmetic, in the same coordinate order, as ls_retry_row
            const float tn = t_i[pp] * a.shrink;
            t_i[pp] = tn;
            float dsum = 0.0f;
#pragma unroll
            for (int c4 = 0; c4 < DP / 4; ++c4) {
              if (4 * c4 < d) {
                const float4 xo = XS[c4 * PTILE + col], pv = PS[c4 * PTILE + col], gv = GS[c4 * PTILE + col];
                float4 xn = make_float4(0.f, 0.f, 0.f, 0.f);
                { xn.x = clipf(fmaf(tn, pv.x, xo.x), a.lo[4 * c4], a.hi[4 * c4]); dsum = fmaf(-gv.x, xn.x - xo.x, dsum); }
                if (4 * c4 + 1 < d) { xn.y = clipf(fmaf(tn, pv.y, xo.y), a.lo[4 * c4 + 1], a.hi[4 * c4 + 1]); dsum = fmaf(-gv.y, xn.y - xo.y, dsum); }
                if (4 * c4 + 2 < d) { xn.z = clipf(fmaf(tn, pv.z, xo.z), a.lo[4 * c4 + 2], a.hi[4 * c4 + 2]); dsum = fmaf(-gv.z, xn.z - xo.z, dsum); }
                if (4 * c4 + 3 < d) { xn.w = clipf(fmaf(tn, pv.w, xo.w), a.lo[4 * c4 + 3], a.hi[4 * c4 + 3]); dsum = fmaf(-gv.w, xn.w - xo.w, dsum); }
                sm.pts[c4 * PTILE + col] = xn;            // own column: read only by this thread in eval_tile
              }
            }
            dec_i[pp] = dsum;
          }
        } else if (retry) {
          const float tn = a.tcur[i] * a.shrink;
          a.tcur[i] = tn;
          a.dec[i] = ls_retry_row(a, i, d, tn);          // rewrites x_t of sample i (read back by this thread only)
        }
        valid[pp] = retry;                                // PT_LS_ALL: the sample stays in its tile slot
        again |= retry;
      }
    }
    if (a.mode != PT_LS_ALL) break;
    if (!__syncthreads_or(again)) break;                  // also orders this round's reads of the staged points before the next staging
  }
  if (a.mode == PT_LS_ALL) {
    nev = (unsigned int)warp_sum_u(nev);
    if ((t & 31) == 0 && nev) atomicAdd(&a.evals[EV_LS], (unsigned long long)nev);
  } else if (t == 0) {
    atomicAdd(&a.evals[a.mode == PT_CENTRE ? EV_INIT : EV_LS], (unsigned long long)min(PTILE, cnt - first));
  }
}

struct HlcArgs {
  const int32_t *list;       // explore list (not stuck, not removed), ascending
  const int32_t *count;
  int32_t max_count, d, M, cycle, iter, baseline;
  float *x, *ghat, *hlc_f;
  const float *lo, *hi;
  const float *sigma_dev;    // ctrl->sigma_eff (caller's sigma_s or the auto-estimate)
  float eta;
  uint64_t seed;
  unsigned long long *evals;
};

// ---- Hands Like Clouds: ghat = (1/(M sigma)) sum_k (f(x + sigma u_k) - b) u_k, x <- clip(x + eta ghat) --
// (Eq. 9; north_star (e); R-11.)  Point p of the tile = (sample p / M,
// draw p % M).  The normals u_k are generated in-thread from Philox (tag HLC_U, sequence index k d + j)
// and kept in shared memory; the perturbed point is staged next to them.
constexpr int HLC_MAX_SPT = 32;
template <int OBJ, int DP>
__global__ void __launch_bounds__(NT, 2) k_hlc(const DevObj o, const HlcArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const EvalSmem sm = carve_smem<DP>(smem_raw, o.kc * o.rec);
  float4 *U = reinterpret_cast<float4 *>(sm.extra);                 // [DP/4][PTILE] normals
  float *fvs = reinterpret_cast<float *>(U + (DP / 4) * PTILE);     // [PTILE] values
  const int t = threadIdx.x, d = a.d, M = a.M;
  const float sigma = *a.sigma_dev;
  if (sigma == 0.0f) return;                       // no spread among the unfrozen samples: nobody moves (R-18)
  const int spt = min(PTILE / M, HLC_MAX_SPT);
  const int cnt = a.count ? *a.count : a.max_count;
  const int first = blockIdx.x * spt;
  if (first >= cnt) return;
  if (t == 0) { mbar_init(&sm.bar[0], 1); mbar_init(&sm.bar[1], 1); mbar_fence_init(); }
  const bool vec = (d & 3) == 0;
  int idx[PPT], kk[PPT]; bool valid[PPT];
#pragma unroll
  for (int pp = 0; pp < PPT; ++pp) {
    const int p = pp * NT + t, s = p / M;
    kk[pp] = p - s * M;
    valid[pp] = (s < spt) && (first + s < cnt);
    idx[pp] = valid[pp] ? a.list[first + s] : 0;
    if (valid[pp]) {
      const float *row = a.x + (size_t)idx[pp] * d;
      const uint32_t tg = rng_tag(5, a.iter, PUR_HLC_U);
      float z0 = 0.f, z1 = 0.f, z2 = 0.f, z3 = 0.f;
      const uint32_t n0 = (uint32_t)kk[pp] * (uint32_t)d;
      uint32_t cur_blk = 0xffffffffu;
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        const float4 xv = ld_row4(row, c4, d, vec);
        float4 uv = make_float4(0.f, 0.f, 0.f, 0.f), pv = xv;
#pragma unroll
        for (int l = 0; l < 4; ++l) {
          const int j = 4 * c4 + l;
          if (j < d) {
            const uint32_t n = n0 + (uint32_t)j;
            if ((n >> 2) != cur_blk) {
              cur_blk = n >> 2;
              const uint4 w = philox_block(a.seed, cur_blk, (uint32_t)idx[pp], (uint32_t)a.cycle, tg);
              box_muller(w.x, w.y, z0, z1);
              box_muller(w.z, w.w, z2, z3);
            }
            const uint32_t ln = n & 3u;
            const float u = ln == 0u ? z0 : (ln == 1u ? z1 : (ln == 2u ? z2 : z3));
            set4(uv, l, u);
            set4(pv, l, fmaf(sigma, u, get4(xv, l)));   // evaluation points are not clipped (R-12)
          }
        }
        U[c4 * PTILE + p] = uv;
        sm.pts[c4 * PTILE + p] = pv;
      }
    } else {
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        U[c4 * PTILE + p] = make_float4(0.f, 0.f, 0.f, 0.f);
        sm.pts[c4 * PTILE + p] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
  }
  __syncthreads();
  uint32_t use = 0;
  float fv[PPT];
  eval_tile<OBJ, DP>(o, sm, t, use, fv);
#pragma unroll
  for (int pp = 0; pp < PPT; ++pp) {
    float val = 0.0f;
    if (valid[pp]) {
      val = fv[pp] + eval_noise(o.sigma_noise, a.seed, a.cycle, idx[pp], 5, a.iter, kk[pp]);
      a.hlc_f[(size_t)idx[pp] * M + kk[pp]] = val;
    }
    fvs[pp * NT + t] = val;
  }
  __syncthreads();
  const int nval = min(spt, cnt - first);
  for (int item = t; item < nval * d; item += NT) {
    const int s = item / d, j = item - s * d;
    const int i = a.list[first + s];
    float b = 0.0f;
    if (a.baseline) {   // (f / M = f * (1 / M) exactly when M is a power of two: M multiplications instead of M divisions per item)
      const bool m_pow2 = (M & (M - 1)) == 0;
      const float inv_m = 1.0f / (float)M;
      for (int k = 0; k < M; ++k) b += m_pow2 ? fvs[s * M + k] * inv_m : fvs[s * M + k] / (float)M;
    }
    float acc = 0.0f;
    for (int k = 0; k < M; ++k) acc = fmaf(fvs[s * M + k] - b, get4(U[(j >> 2) * PTILE + s * M + k], j & 3), acc);
    const float gh = acc / ((float)M * sigma);
    a.ghat[(size_t)i * d + j] = gh;
    // x_j of the centre = staged point minus sigma u is not exact; re-read the row (written only here)
    const float xo = a.x[(size_t)i * d + j];
    a.x[(size_t)i * d + j] = clipf(fmaf(a.eta, gh, xo), a.lo[j], a.hi[j]);
  }
  if (t == 0) atomicAdd(&a.evals[EV_HLC], (unsigned long long)nval * (unsigned long long)M);
}

// ---- launchers (one set per objective id) --------------------------------------------------------------
template <int OBJ, int DP>
inline cudaError_t configure_one() {
  cudaError_t e;
  const int big = 200 * 1024;
  e = cudaFuncSetAttribute(k_eval_fd<OBJ, DP>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(k_eval_points<OBJ, DP>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_hlc<OBJ, DP>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
}
template <int OBJ>
cudaError_t configure_obj() {
  cudaError_t e = configure_one<OBJ, 8>();
  if (e != cudaSuccess) return e;
  e = configure_one<OBJ, 32>();
  if (e != cudaSuccess) return e;
  return configure_one<OBJ, 64>();
}

inline size_t hlc_extra_bytes(int DP) { return (size_t)(DP / 4) * PTILE * 16 + PTILE * 4; }

template <int OBJ>
cudaError_t launch_fd_obj(const DevObj &o, const FdArgs &a, int grid, cudaStream_t st) {
  const size_t sh = eval_smem_bytes(o, 0);
  switch (o.DP) {
    case 8: k_eval_fd<OBJ, 8><<<grid, NT, sh, st>>>(o, a); break;
    case 32: k_eval_fd<OBJ, 32><<<grid, NT, sh, st>>>(o, a); break;
    default: k_eval_fd<OBJ, 64><<<grid, NT, sh, st>>>(o, a); break;
  }
  return cudaGetLastError();
}
inline size_t ls_rows_bytes(int DP) { return (size_t)3 * (DP / 4) * PTILE * 16; }
template <int OBJ>
cudaError_t launch_pt_obj(const DevObj &o, const PtArgs &a, int grid, cudaStream_t st) {
  const size_t sh = eval_smem_bytes(o, a.rows_in_smem ? ls_rows_bytes(o.DP) : 0);
  switch (o.DP) {
    case 8: k_eval_points<OBJ, 8><<<grid, NT, sh, st>>>(o, a); break;
    case 32: k_eval_points<OBJ, 32><<<grid, NT, sh, st>>>(o, a); break;
    default: k_eval_points<OBJ, 64><<<grid, NT, sh, st>>>(o, a); break;
  }
  return cudaGetLastError();
}
template <int OBJ>
cudaError_t launch_hlc_obj(const DevObj &o, const HlcArgs &a, int grid, cudaStream_t st) {
  const size_t sh = eval_smem_bytes(o, hlc_extra_bytes(o.DP));
  switch (o.DP) {
    case 8: k_hlc<OBJ, 8><<<grid, NT, sh, st>>>(o, a); break;
    case 32: k_hlc<OBJ, 32><<<grid, NT, sh, st>>>(o, a); break;
    default: k_hlc<OBJ, 64><<<grid, NT, sh, st>>>(o, a); break;
  }
  return cudaGetLastError();
}

// per-objective entry points defined in chisao_eval_obj.cu
#define CHISAO_DECL_OBJ(ID)                                                                        \
  cudaError_t launch_fd_obj_##ID(const DevObj &, const FdArgs &, int, cudaStream_t);                \
  cudaError_t launch_pt_obj_##ID(const DevObj &, const PtArgs &, int, cudaStream_t);                \
  cudaError_t launch_hlc_obj_##ID(const DevObj &, const HlcArgs &, int, cudaStream_t);              \
  cudaError_t configure_obj_##ID();
CHISAO_DECL_OBJ(0) CHISAO_DECL_OBJ(1) CHISAO_DECL_OBJ(2) CHISAO_DECL_OBJ(3) CHISAO_DECL_OBJ(4) CHISAO_DECL_OBJ(5)

}  // namespace chisao
