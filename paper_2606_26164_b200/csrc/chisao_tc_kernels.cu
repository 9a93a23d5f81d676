// chisao_tc_kernels.cu -- the three evaluation kernels (FD stencil, one point per sample, Hands Like Clouds)
// on the tensor-core evaluator of chisao_tc.cuh, for GMM_FULL and QUAD at 32 < d <= 64 and RFF at d <= 32, K <= 256.  Same arguments, same
// noise slots, same epilogues as the FFMA kernels of chisao_eval_kernels.cuh; one point per compute thread, 256
// points per CTA (two groups of 128 ping-pong on the tensor pipe) plus one warp that streams the parameters.  Citations: PAPER.md:62, :555 (FD), :75-82 (line search), :113-120 + Eq. 9 :577 (HLC), Eq. 6 :126.
#include "chisao_eval_kernels.cuh"
#include "chisao_tc.cuh"

namespace chisao {

__device__ __forceinline__ void compute_sync() { asm volatile("bar.sync 3, %0;" ::"n"(TC_PTS) : "memory"); }

__device__ __forceinline__ void tc_load_row(const float *row, int d, bool vec, float (&x)[TC_D]) {
#pragma unroll
  for (int c4 = 0; c4 < TC_D / 4; ++c4) {
    const float4 v = ld_row4(row, c4, d, vec);
    x[4 * c4] = v.x; x[4 * c4 + 1] = v.y; x[4 * c4 + 2] = v.z; x[4 * c4 + 3] = v.w;
  }
}

// thread t of group t >> 7 -> (sample (t & 127) / 2d of the group, slot (t & 127) % 2d); slot 2j = x + h e_j,
// 2j + 1 = x - h e_j.  The 2d stencil points of a sample never straddle the two groups of 128 points: in the QUAD and RFF
// forms the groups run unsynchronised (one may be a tile ahead of the other), and FD_ANTI rewrites the sample's row
// in place from the finish of the group that owns it -- a row shared by both groups could be read half-updated.
__host__ __device__ inline int fd_tc_samples_per_tile(int d) { return 2 * (TC_GROUP / (2 * d)); }
struct FdCtx { int i; float xj, xp; bool valid; };
template <int OBJ>
__global__ void __launch_bounds__(TC_THREADS, 1) k_eval_fd_tc(const TcObj o, const FdArgs a) {
  extern __shared__ __align__(1024) unsigned char tc_smem_raw[];
  const TcSmem sm = tc_carve(tc_smem_raw);
  const int t = threadIdx.x, d = a.d;
  const int spg = TC_GROUP / (2 * d), spt = 2 * spg;
  const int cnt = a.count ? *a.count : a.max_count;
  const int ntiles = (cnt + spt - 1) / spt;
  if (blockIdx.x == 0 && t == 0 && a.zero_cnt) *a.zero_cnt = 0;
  if ((int)blockIdx.x >= ntiles) return;
  tc_begin<OBJ>(sm, t);
  const int tl = t & (TC_GROUP - 1), sg = tl / (2 * d), slot = tl - sg * 2 * d, j = slot >> 1;
  const int s = (t < TC_PTS && sg < spg) ? (t >> 7) * spg + sg : spt;   // s >= spt: idle lane (also the loader / issuer warps)
  auto load = [&](int tile, float (&x)[TC_D]) -> FdCtx {
    FdCtx c;
    const int first = tile * spt;
    c.valid = (s < spt) && (first + s < cnt);
    c.i = c.valid ? (a.list ? a.list[first + s] : first + s) : 0;
    // the CTA's next tile: its worklist entry is pulled into L1 now, so that the dependent load in front of the row
    // loads is a hit by then
    if (OBJ != CHISAO_OBJ_GMM_FULL && a.list && s < spt) {   // (GMM_FULL fetches its next tile a whole tile ahead)
      const int nf = (tile + (int)gridDim.x) * spt + s;
      if (nf < cnt) asm volatile("prefetch.global.L1 [%0];" ::"l"(a.list + nf));
    }
    c.xj = 0.f; c.xp = 0.f;
    if (c.valid) {
      const float *row = a.X + (size_t)c.i * d;
      tc_load_row(row, d, (d & 3) == 0, x);
      c.xj = row[j];
      c.xp = (slot & 1) ? c.xj - a.h : c.xj + a.h;
      // replace coordinate j by compare-and-select over the whole row: every lane runs the same straight-line code (a
      // dynamically indexed register array would be lowered to a branch tree over j, and the warp-collective tcgen05
      // instructions of the evaluator need every lane on the same path), and nothing waits for the row here -- the
      // global loads stay in flight until the evaluator first touches x
      if constexpr (OBJ != CHISAO_OBJ_GMM_FULL) {
#pragma unroll
        for (int q = 0; q < TC_D; ++q) x[q] = (q == j) ? c.xp : x[q];
      } else {
        // GMM_FULL (the row is consumed within the same pair iteration anyway; 64 selects cost registers there): the
        // thread's own row goes through shared memory and comes back with coordinate j patched
        float *own = reinterpret_cast<float *>(sm.scratch()) + t * 68;
#pragma unroll
        for (int c4 = 0; c4 < TC_D / 4; ++c4)
          *reinterpret_cast<float4 *>(own + 4 * c4) = make_float4(x[4 * c4], x[4 * c4 + 1], x[4 * c4 + 2], x[4 * c4 + 3]);
        own[j] = c.xp;                       // same thread writes and reads its row: program order suffices
#pragma unroll
        for (int c4 = 0; c4 < TC_D / 4; ++c4) {
          const float4 v = *reinterpret_cast<const float4 *>(own + 4 * c4);
          x[4 * c4] = v.x; x[4 * c4 + 1] = v.y; x[4 * c4 + 2] = v.z; x[4 * c4 + 3] = v.w;
        }
      }
    } else {
#pragma unroll
      for (int c = 0; c < TC_D; ++c) x[c] = 0.f;
    }
    return c;
  };
  auto finish = [&](int tile, float f, const FdCtx &c) {
    if (c.valid) f += eval_noise(o.sigma_noise, a.seed, a.cycle, c.i, a.phase, a.iter, a.slot_off + 1 + slot);
    // partner lane holds the other sign of the same coordinate
    const float fo = __shfl_xor_sync(0xffffffffu, f, 1);
    const float xo = __shfl_xor_sync(0xffffffffu, c.xp, 1);
    if (c.valid && !(slot & 1)) {
      const float g = (f - fo) / ((c.xp - c.xj) + (c.xj - xo));
      if (a.mode == FD_GRAD) {
        a.g_out[(size_t)c.i * d + j] = g;
      } else {   // Eq. 6
        const float vo = (a.iter == 1) ? 0.0f : a.v[(size_t)c.i * d + j];
        const float vn = fmaf(a.mu, vo, -a.alpha * g);
        a.v[(size_t)c.i * d + j] = vn;
        a.x[(size_t)c.i * d + j] = clipf(c.xj + vn, a.lo[j], a.hi[j]);
      }
    }
    if (t == 0) atomicAdd(&a.evals[a.counter], (unsigned long long)min(spt, cnt - tile * spt) * 2ull * d);
  };
  tc_run<OBJ>(o, sm, t, ntiles, load, finish);
  tc_teardown(sm, t);
}

struct PtCtx { int i; bool valid; };
template <int OBJ>
__global__ void __launch_bounds__(TC_THREADS, 1) k_eval_points_tc(const TcObj o, const PtArgs a) {
  extern __shared__ __align__(1024) unsigned char tc_smem_raw[];
  const TcSmem sm = tc_carve(tc_smem_raw);
  const int t = threadIdx.x, d = a.d;
  const int cnt = a.count ? *a.count : a.max_count;
  const int ntiles = (cnt + TC_PTS - 1) / TC_PTS;
  if (blockIdx.x == 0 && t == 0 && a.zero_cnt) *a.zero_cnt = 0;
  if ((int)blockIdx.x >= ntiles) return;
  tc_begin<OBJ>(sm, t);
  if constexpr (OBJ != CHISAO_OBJ_GMM_FULL) {
    if (a.mode == PT_LS_ALL) {
      // every trial b = 0 .. ls_max of the CTA's 256 worklist entries in one launch (tc_rounds): round r = trial b
      const int e = (int)blockIdx.x * TC_PTS + t;
      bool active = (t < TC_PTS) && (e < cnt);
      const int i = active ? a.list[e] : 0;
      unsigned int nev = 0;
      auto load = [&](int, float (&x)[TC_D]) {
        if (active) tc_load_row(a.X + (size_t)i * d, d, (d & 3) == 0, x);
        else {
#pragma unroll
          for (int k = 0; k < TC_D; ++k) x[k] = 0.f;
        }
      };
      auto finish = [&](int b, float fv) -> bool {
        bool accept = false, retry = false;
        float val = 0.f;
        if (active) {
          val = fv + eval_noise(o.sigma_noise, a.seed, a.cycle, i, 1, a.iter, 2 * d + 1 + b);
          accept = ls_accept(val, a.f[i], a.dec[i], a.c1);
          retry = !accept && (b < a.ls_max);
          nev += 1u;
        }
        const int sa = warp_append(a.fd_cnt, accept);
        if (accept) { a.fd_list[sa] = i; a.ls_b[i] = b; a.ft[i] = val; }
        if (retry) {
          const float tn = a.tcur[i] * a.shrink;
          a.tcur[i] = tn;
          a.dec[i] = ls_retry_row(a, i, d, tn);            // rewrites x_t of sample i (read back by this thread only)
        }
        active = retry;
        return retry;
      };
      tc_rounds<OBJ>(o, sm, t, load, finish);
      if (t < TC_PTS) {
        nev = warp_sum_u(nev);
        if ((t & 31) == 0 && nev) atomicAdd(&a.evals[EV_LS], (unsigned long long)nev);
      }
      tc_teardown(sm, t);
      return;
    }
  }
  auto load = [&](int tile, float (&x)[TC_D]) -> PtCtx {
    PtCtx c;
    const int e = tile * TC_PTS + t;
    c.valid = e < cnt;
    c.i = c.valid ? (a.list ? a.list[e] : e) : 0;
    if (c.valid) tc_load_row(a.X + (size_t)c.i * d, d, (d & 3) == 0, x);
    else {
#pragma unroll
      for (int k = 0; k < TC_D; ++k) x[k] = 0.f;
    }
    return c;
  };
  auto finish = [&](int tile, float fv, const PtCtx &c) {
    const int i = c.i;
    bool accept = false, retry = false;
    float val = 0.f;
    if (c.valid) {
      if (a.mode == PT_CENTRE) {
        a.f[i] = fv + eval_noise(o.sigma_noise, a.seed, a.cycle, i, 1, 0, 0);
      } else {
        val = fv + eval_noise(o.sigma_noise, a.seed, a.cycle, i, 1, a.iter, 2 * d + 1 + a.b);
        accept = ls_accept(val, a.f[i], a.dec[i], a.c1);
        retry = !accept && (a.b < a.ls_max);
      }
    }
    if (a.mode == PT_LS) {
      const int sa = warp_append(a.fd_cnt, accept);
      if (accept) { a.fd_list[sa] = i; a.ls_b[i] = a.b; a.ft[i] = val; }
      const int sr = warp_append(a.next_cnt, retry);
      if (retry) {
        a.next_list[sr] = i;
        const float tn = a.tcur[i] * a.shrink;
        a.tcur[i] = tn;
        a.dec[i] = ls_retry_row(a, i, d, tn);
      }
    }
    if (t == 0)
      atomicAdd(&a.evals[a.mode == PT_CENTRE ? EV_INIT : EV_LS], (unsigned long long)min(TC_PTS, cnt - tile * TC_PTS));
  };
  tc_run<OBJ>(o, sm, t, ntiles, load, finish);
  tc_teardown(sm, t);
}

// the d normals of draw k of sample i (Philox tag HLC_U, sequence index k d + j; R-15)
__device__ __forceinline__ void hlc_normals(uint64_t seed, int i, int cycle, int iter, int k, int d, float (&u)[TC_D]) {
  const uint32_t tg = rng_tag(5, iter, PUR_HLC_U);
  const uint32_t n0 = (uint32_t)k * (uint32_t)d;
  if ((d & 3) == 0) {   // the draw's d normals are d / 4 whole Philox blocks: independent chains the scheduler can interleave
#pragma unroll
    for (int b = 0; b < TC_D / 4; ++b) {
      if (4 * b < d) {    // warp-uniform
        const uint4 w = philox_block(seed, (n0 >> 2) + (uint32_t)b, (uint32_t)i, (uint32_t)cycle, tg);
        box_muller(w.x, w.y, u[4 * b], u[4 * b + 1]);
        box_muller(w.z, w.w, u[4 * b + 2], u[4 * b + 3]);
      } else {
        u[4 * b] = 0.f; u[4 * b + 1] = 0.f; u[4 * b + 2] = 0.f; u[4 * b + 3] = 0.f;
      }
    }
    return;
  }
  float z0 = 0.f, z1 = 0.f, z2 = 0.f, z3 = 0.f;
  uint32_t cur = 0xffffffffu;
#pragma unroll
  for (int j = 0; j < TC_D; ++j) {
    float v = 0.f;
    if (j < d) {
      const uint32_t n = n0 + (uint32_t)j;
      if ((n >> 2) != cur) {
        cur = n >> 2;
        const uint4 w = philox_block(seed, cur, (uint32_t)i, (uint32_t)cycle, tg);
        box_muller(w.x, w.y, z0, z1);
        box_muller(w.z, w.w, z2, z3);
      }
      const uint32_t ln = n & 3u;
      v = ln == 0u ? z0 : (ln == 1u ? z1 : (ln == 2u ? z2 : z3));
    }
    u[j] = v;
  }
}

// Hands Like Clouds on the tensor-core evaluator: point t of the tile = (sample t / M, draw t % M), M <= 128
struct HlcCtx { int i; bool valid; };
template <int OBJ>
__global__ void __launch_bounds__(TC_THREADS, 1) k_hlc_tc(const TcObj o, const HlcArgs a) {
  extern __shared__ __align__(1024) unsigned char tc_smem_raw[];
  const TcSmem sm = tc_carve(tc_smem_raw);
  const int t = threadIdx.x, d = a.d, M = a.M;
  const float sigma = *a.sigma_dev;
  if (sigma == 0.0f) return;                       // no spread among the unfrozen samples: nobody moves (R-18)
  const int spt = min(TC_PTS / M, HLC_MAX_SPT);
  const int cnt = a.count ? *a.count : a.max_count;
  const int ntiles = (cnt + spt - 1) / spt;
  if ((int)blockIdx.x >= ntiles) return;
  tc_begin<OBJ>(sm, t);
  const int s = t / M, k = t - s * M;
  auto load = [&](int tile, float (&x)[TC_D]) -> HlcCtx {
    HlcCtx c;
    const int first = tile * spt;
    c.valid = (s < spt) && (first + s < cnt);
    c.i = c.valid ? a.list[first + s] : 0;
    if (c.valid) {
      float u[TC_D];
      hlc_normals(a.seed, c.i, a.cycle, a.iter, k, d, u);
      tc_load_row(a.x + (size_t)c.i * d, d, (d & 3) == 0, x);
#pragma unroll
      for (int q = 0; q < TC_D; ++q) x[q] = fmaf(sigma, u[q], x[q]);   // evaluation points are not clipped (R-12)
    } else {
#pragma unroll
      for (int q = 0; q < TC_D; ++q) x[q] = 0.f;
    }
    return c;
  };
  // Positions are only written by the tile that owns the sample, after every point of that tile has been read
  // (load of the tile precedes its finish); tiles own disjoint samples.
  auto finish = [&](int tile, float val, const HlcCtx &c) {
    const int first = tile * spt, i = c.i;
    compute_sync();                        // the previous tile's estimate has been read out of the scratch
    float *Us = reinterpret_cast<float *>(sm.scratch());        // [256][65] normals (scratch is 72 KB)
    float *fvs = Us + TC_PTS * 65;                              // [256] values
    if (c.valid) {
      val += eval_noise(o.sigma_noise, a.seed, a.cycle, i, 5, a.iter, k);
      a.hlc_f[(size_t)i * M + k] = val;
      float u[TC_D];
      hlc_normals(a.seed, i, a.cycle, a.iter, k, d, u);
#pragma unroll
      for (int q = 0; q < TC_D; ++q) Us[t * 65 + q] = u[q];
    } else {
      val = 0.f;
    }
    fvs[t] = val;
    compute_sync();
    const int nval = min(spt, cnt - first);
    for (int item = t; item < nval * d; item += TC_PTS) {
      const int ss = item / d, j = item - ss * d;
      const int ii = a.list[first + ss];
      float b = 0.0f;
      if (a.baseline) for (int kk = 0; kk < M; ++kk) b += fvs[ss * M + kk] / (float)M;
      float acc = 0.0f;
      for (int kk = 0; kk < M; ++kk) acc = fmaf(fvs[ss * M + kk] - b, Us[(ss * M + kk) * 65 + j], acc);
      const float gh = acc / ((float)M * sigma);
      a.ghat[(size_t)ii * d + j] = gh;
      const float xo = a.x[(size_t)ii * d + j];
      a.x[(size_t)ii * d + j] = clipf(fmaf(a.eta, gh, xo), a.lo[j], a.hi[j]);
    }
    if (t == 0) atomicAdd(&a.evals[EV_HLC], (unsigned long long)nval * (unsigned long long)M);
  };
  tc_run<OBJ>(o, sm, t, ntiles, load, finish);
  tc_teardown(sm, t);
}

// ---- launchers ------------------------------------------------------------------------------------------------
static int g_tc_sms = 148;
static inline int tc_grid(int obj_id, int ntiles) {   // persistent CTAs, one per SM
  (void)obj_id;
  return ntiles > g_tc_sms ? g_tc_sms : ntiles;
}
cudaError_t tc_configure() {
  cudaError_t e;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
    g_tc_sms = sms;
#define CFG(K) if ((e = cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM_BYTES)) != cudaSuccess) return e;
  CFG(k_eval_fd_tc<CHISAO_OBJ_GMM_FULL>) CFG(k_eval_fd_tc<CHISAO_OBJ_QUAD>)
  CFG(k_eval_points_tc<CHISAO_OBJ_GMM_FULL>) CFG(k_eval_points_tc<CHISAO_OBJ_QUAD>)
  CFG(k_hlc_tc<CHISAO_OBJ_GMM_FULL>) CFG(k_hlc_tc<CHISAO_OBJ_QUAD>)
  CFG(k_eval_fd_tc<CHISAO_OBJ_RFF>) CFG(k_eval_points_tc<CHISAO_OBJ_RFF>) CFG(k_hlc_tc<CHISAO_OBJ_RFF>)
#undef CFG
  return cudaSuccess;
}
cudaError_t launch_fd_tc(int obj_id, const TcObj &o, const FdArgs &a, int n_samples, cudaStream_t st) {
  const int spt = fd_tc_samples_per_tile(a.d);
  const int grid = tc_grid(obj_id, (n_samples + spt - 1) / spt);
  if (obj_id == CHISAO_OBJ_QUAD) k_eval_fd_tc<CHISAO_OBJ_QUAD><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else if (obj_id == CHISAO_OBJ_RFF) k_eval_fd_tc<CHISAO_OBJ_RFF><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else k_eval_fd_tc<CHISAO_OBJ_GMM_FULL><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  return cudaGetLastError();
}
cudaError_t launch_pt_tc(int obj_id, const TcObj &o, const PtArgs &a, int n_samples, cudaStream_t st) {
  const int ntiles = (n_samples + TC_PTS - 1) / TC_PTS;
  const int grid = (a.mode == PT_LS_ALL) ? ntiles : tc_grid(obj_id, ntiles);   // tile-local rounds: one tile per CTA
  if (obj_id == CHISAO_OBJ_QUAD) k_eval_points_tc<CHISAO_OBJ_QUAD><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else if (obj_id == CHISAO_OBJ_RFF) k_eval_points_tc<CHISAO_OBJ_RFF><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else k_eval_points_tc<CHISAO_OBJ_GMM_FULL><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  return cudaGetLastError();
}
cudaError_t launch_hlc_tc(int obj_id, const TcObj &o, const HlcArgs &a, int n_samples, cudaStream_t st) {
  const int spt = TC_PTS / a.M < HLC_MAX_SPT ? TC_PTS / a.M : HLC_MAX_SPT;
  const int grid = tc_grid(obj_id, (n_samples + spt - 1) / spt);
  if (obj_id == CHISAO_OBJ_QUAD) k_hlc_tc<CHISAO_OBJ_QUAD><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else if (obj_id == CHISAO_OBJ_RFF) k_hlc_tc<CHISAO_OBJ_RFF><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else k_hlc_tc<CHISAO_OBJ_GMM_FULL><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  return cudaGetLastError();
}

}  // namespace chisao
