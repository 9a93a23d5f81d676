// chisao_resident.cuh -- the history-RESIDENT form of Phase 1 (Eq. 2; readings R-4, R-5, R-6): one launch
// runs L-BFGS iterations it0 .. it1 for the samples of a CTA, which keeps them for the whole pass -- samples are
// independent during Phase 1, so no grid-wide step is needed.  The (s, y) history of a sample never
// touches HBM during the pass: it lives in REGISTERS (thread (sample, coordinate j) holds coordinate j of every stored
// pair; BASELINE.json north_star: "L-BFGS (s,y) histories sit in SMEM or registers, with ... HBM traffic for history
// spill at large N" -- the spill form is chisao_lbfgs.cu).  Dots are segmented warp shuffles over the d lanes of a
// sample (d a power of two <= 32); objective evaluations go through the same evaluator as everywhere else
// (eval_tile: the line-search trial of every sample of the CTA as one tile, the 2d stencil points of every sample as
// one tile), with the objective's parameters resident in shared memory after the first call.
//
// Chosen at chisao_init for the FP32-FMA evaluators when d is 1, 2, 4, 8, 16 or 32, the parameters fit one chunk and
// m <= 16 (C1, C2); CHISAO_OPT_LBFGS_RESIDENT switches it.  Inside a cycle the launch also does what precedes and follows
// the pass: release-all + f, g at the start positions (it0 = 0), and Phase 2's per-sample partials at the end.
#pragma once
#include "chisao_eval_kernels.cuh"

namespace chisao {

struct ResArgs {
  State s;
  Hyper h;
  int32_t cycle;
  int32_t it0, it1;          // iterations it0 .. it1 (1-based); it0 = 0: release + first evaluation, then 1 .. it1
  int32_t write_diag;        // stand-alone unit: direction, trial point and accepted-trial index go to the state like the spill form's
  int32_t stick_partials;    // end of a pass inside a cycle: ||grad f||_inf per sample and the f_max partials of Phase 2
};

template <int D>
__device__ __forceinline__ float seg_sum(float v, int d) {   // sum over the d aligned lanes of a sample (all 32 lanes call)
#pragma unroll
  for (int o = D / 2; o > 0; o >>= 1) if (o < d) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
template <int D>
__device__ __forceinline__ float seg_max(float v, int d) {
#pragma unroll
  for (int o = D / 2; o > 0; o >>= 1) if (o < d) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

template <int OBJ, int DP, int MM>
__global__ void __launch_bounds__(NT, 2) k_lbfgs_resident(const DevObj o, const ResArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const EvalSmem sm = carve_smem<DP>(smem_raw, o.kc * o.rec);
  float *xrow = sm.extra;                 // [NT] the rows the stencil is centred on: sample slot sl, coordinate j at sl d + j
  float *fval = xrow + NT;                // [NT] one value per sample slot
  __shared__ unsigned int sh_ev[3];
  const State &s = a.s;
  const Hyper &h = a.h;
  const int t = threadIdx.x, d = s.d, m = s.m, N = s.N;
  const int spt = NT / d, sl = t / d, j = t - sl * d;
  const int i = blockIdx.x * spt + sl;
  const bool in = i < N;
  const size_t e = (size_t)(in ? i : 0) * d + j;
  if (t == 0) { mbar_init(&sm.bar[0], 1); mbar_init(&sm.bar[1], 1); mbar_fence_init(); }
  if (t < 3) sh_ev[t] = 0u;
  for (int c = t; c < (DP / 4) * PTILE; c += NT) sm.pts[c] = make_float4(0.f, 0.f, 0.f, 0.f);   // padding coordinates stay zero
  __syncthreads();
  const float lo = s.lo[j], hi = s.hi[j];
  float *pcol = reinterpret_cast<float *>(sm.pts + (j >> 2) * PTILE + sl) + (j & 3);   // coordinate j of the point in column sl
  uint32_t use = 0;
  unsigned int n_init = 0, n_ls = 0, n_fd = 0;   // evaluations counted by the j = 0 thread of a sample

  // central finite differences at the rows in xrow (R-1), as k_eval_fd stages and forms them;
  // `want`: the sample needs the gradient (the others ride along in the tile)
  auto fd_gradient = [&](int iter, float xj) -> float {
    const float xph = xj + h.fd_h, xmh = xj - h.fd_h;
#pragma unroll
    for (int c4 = 0; c4 < DP / 4; ++c4) {
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (4 * c4 < d) {
        const float *r = xrow + sl * d + 4 * c4;
        v.x = r[0];
        if (4 * c4 + 1 < d) v.y = r[1];
        if (4 * c4 + 2 < d) v.z = r[2];
        if (4 * c4 + 3 < d) v.w = r[3];
      }
      float4 vp = v, vm = v;
      if (c4 == (j >> 2)) { set4(vp, j & 3, xph); set4(vm, j & 3, xmh); }
      sm.pts[c4 * PTILE + t] = vp;
      sm.pts[c4 * PTILE + NT + t] = vm;
    }
    __syncthreads();
    float fv[PPT];
    eval_tile<OBJ, DP>(o, sm, t, use, fv);
    const float fp = fv[0] + eval_noise(o.sigma_noise, h.seed, a.cycle, i, 1, iter, 1 + 2 * j);
    const float fm = fv[1] + eval_noise(o.sigma_noise, h.seed, a.cycle, i, 1, iter, 2 + 2 * j);
    __syncthreads();                          // every thread has read its staged points: the tile may be rewritten
    return (fp - fm) / ((xph - xj) + (xj - xmh));
  };
  // one point per sample: coordinate j of the sample's point goes to column sl, the value comes back to all d lanes
  auto point_value = [&](float xj) -> float {
    *pcol = xj;
    __syncthreads();
    float fv[PPT];
    eval_tile<OBJ, DP>(o, sm, t, use, fv);
    if (t < spt) fval[t] = fv[0];
    __syncthreads();
    return fval[sl];
  };

  // ---- state of the sample into registers --------------------------------------------------------------------------
  float x = in ? s.x[e] : 0.f, g = 0.f, f = 0.f;
  int len = 0, stalled = 0;
  float Sr[MM], Yr[MM];
#pragma unroll
  for (int l = 0; l < MM; ++l) { Sr[l] = 0.f; Yr[l] = 0.f; }
  if (a.it0 == 0) {
    // "stuck <- False^N" (Alg. 1), history reset of every Phase 1 (R-5), f and g at the start positions
    if (in && j == 0) { s.stuck[i] = 0; s.removed[i] = 0; s.stalled[i] = 0; }
    const float fc = point_value(x);
    f = fc + eval_noise(o.sigma_noise, h.seed, a.cycle, i, 1, 0, 0);
    xrow[t] = x;
    __syncthreads();
    g = fd_gradient(0, x);
    if (in && j == 0) n_init += 2u * d + 1u;
  } else if (in) {
    f = s.f[i]; g = s.g[e]; len = s.hist_len[i]; stalled = s.stalled[i];
    const int head = s.hist_head[i];
#pragma unroll
    for (int l = 0; l < MM; ++l)
      if (l < len) {
        int ph = head + l; if (ph >= m) ph -= m;
        Sr[l] = s.S[((size_t)ph * s.hplane + (size_t)i * d + j)];
        Yr[l] = s.Y[((size_t)ph * s.hplane + (size_t)i * d + j)];
      }
  }
  if (!in) { g = 0.f; x = 0.f; }

  // ---- the pass ---------------------------------------------------------------------------------------------------------
  for (int it = max(a.it0, 1); it <= a.it1; ++it) {
    const float ginf = seg_max<32>(fabsf(g), d);
    // (i) stationary (Eq. 3's gradient test) or stalled: no work, no evaluations (R-6)
    const bool act = in && !(stalled || !(ginf >= h.eps_grad));
    if (!__syncthreads_or(act)) {            // nobody in this CTA will move again in this pass
      if (a.write_diag && in) { s.p[e] = 0.f; if (j == 0) s.ls_b[i] = -2; }
      break;
    }
    // (ii) two-loop recursion (Nocedal & Wright Alg. 7.4), H0 = (s.y / y.y) I of the newest pair
    const float gam = -g;
    const float gn2 = seg_sum<32>(g * g, d);
    float rho[MM], al[MM];
    float r = gam;
    const int len_read = act ? len : 0;
#pragma unroll
    for (int l = 0; l < MM; ++l) { const float sy = seg_sum<32>(Sr[l] * Yr[l], d); rho[l] = (l < len_read) ? 1.0f / sy : 0.0f; }
#pragma unroll
    for (int l = MM - 1; l >= 0; --l) { al[l] = rho[l] * seg_sum<32>(Sr[l] * r, d); r = fmaf(-al[l], Yr[l], r); }
    float yn = 0.f, rho_n = 1.0f;
#pragma unroll
    for (int l = 0; l < MM; ++l) if (l == len_read - 1) { yn = Yr[l]; rho_n = rho[l]; }
    const float ynyn = seg_sum<32>(yn * yn, d);
    if (len_read > 0) r *= 1.0f / (rho_n * ynyn);
#pragma unroll
    for (int l = 0; l < MM; ++l) { const float beta = rho[l] * seg_sum<32>(Yr[l] * r, d); r = fmaf(al[l] - beta, Sr[l], r); }
    float p = -r;
    const float gp = seg_sum<32>(gam * p, d);
    if (act && len > 0 && !(gp < 0.0f)) len = 0;           // not a descent direction for phi = -f: steepest restart, history cleared
    if (!act || len == 0) p = -gam;
    if (!act) p = 0.f;
    // (iii) first trial step; (iv) projected trial point and the Armijo linear term gamma.(x_t - x)
    float tcur = (len > 0) ? 1.0f : fminf(1.0f, 1.0f / sqrtf(gn2));
    float xt = clipf(fmaf(tcur, p, x), lo, hi);
    float dec = seg_sum<32>(gam * (xt - x), d);
    bool searching = act, accepted = false;
    int bacc = act ? -1 : -2;
    float ft = 0.f;
    for (int b = 0;; ++b) {
      const float fvx = point_value(searching ? xt : x);
      bool retry = false;
      if (searching) {
        const float val = fvx + eval_noise(o.sigma_noise, h.seed, a.cycle, i, 1, it, 2 * d + 1 + b);
        if (j == 0) n_ls += 1u;
        if (ls_accept(val, f, dec, h.ls_c1)) { accepted = true; searching = false; bacc = b; ft = val; }
        else if (b < h.ls_max) { retry = true; tcur *= h.ls_shrink; }
        else searching = false;
      }
      // the shrunk trial point (every lane runs the shuffles; only retrying samples keep the result)
      const float xn = clipf(fmaf(tcur, p, x), lo, hi);
      const float dn = seg_sum<32>(gam * (xn - x), d);
      if (retry) { xt = xn; dec = dn; }
      if (!__syncthreads_or(searching)) break;
    }
    // (vi) gradient at the accepted points (2d evaluations), curvature pair, state
    float gnew = g;
    if (__syncthreads_or(accepted)) {
      xrow[t] = accepted ? xt : x;
      __syncthreads();
      const float gq = fd_gradient(it, accepted ? xt : x);
      if (accepted) { gnew = gq; if (j == 0) n_fd += 2u * d; }
    }
    const float sv = accepted ? xt - x : 0.f, yv = accepted ? g - gnew : 0.f;
    const float sy = seg_sum<32>(sv * yv, d), ss = seg_sum<32>(sv * sv, d), yy = seg_sum<32>(yv * yv, d);
    if (a.write_diag && in) {
      s.p[e] = p;
      if (act) s.xt[e] = xt;
      if (j == 0) s.ls_b[i] = bacc;
    }
    if (accepted) {
      if (sy > 1e-10f * sqrtf(ss) * sqrtf(yy)) {           // store the pair (ring: the oldest is dropped beyond m)
        if (len == m) {
#pragma unroll
          for (int l = 0; l < MM - 1; ++l) if (l < m - 1) { Sr[l] = Sr[l + 1]; Yr[l] = Yr[l + 1]; }
          len = m - 1;
        }
#pragma unroll
        for (int l = 0; l < MM; ++l) if (l == len) { Sr[l] = sv; Yr[l] = yv; }
        len += 1;
      }
      x = xt; g = gnew; f = ft;
    } else if (act) {                                      // (v) no trial accepted
      if (len == 0) stalled = 1; else len = 0;
    }
#pragma unroll
    for (int l = 0; l < MM; ++l) if (l >= len) { Sr[l] = 0.f; Yr[l] = 0.f; }   // cleared slots must not leak into the next dots
  }

  // ---- state back to HBM (logical order: ring head 0) ---------------------------------------------------------------
  if (in) {
    s.x[e] = x; s.g[e] = g;
#pragma unroll
    for (int l = 0; l < MM; ++l)
      if (l < len) { s.S[((size_t)l * s.hplane + (size_t)i * d + j)] = Sr[l]; s.Y[((size_t)l * s.hplane + (size_t)i * d + j)] = Yr[l]; }
    if (j == 0) { s.f[i] = f; s.hist_len[i] = len; s.hist_head[i] = 0; s.stalled[i] = (uint8_t)stalled; }
  }
  if (a.stick_partials) {                                  // Phase 2's partials (what k_ginf_fmax computes)
    const float ag = fabsf(g);
    const bool nan = !(ag == ag);
    const float gi = seg_max<32>(ag, d);
    const float anyn = seg_max<32>(nan ? 1.0f : 0.0f, d);
    float fm = -INFINITY;
    if (in && j == 0) {
      s.ginf[i] = (anyn > 0.f) ? NAN : gi;
      if (fabsf(f) <= 3.0e38f) fm = f;
    }
    fm = warp_max(fm);
    if ((t & 31) == 0 && fm > -INFINITY) atomicMax(&s.ctrl->fmax_enc, enc_ordered(fm));
  }
  // evaluation counters: one atomic per counter and CTA
  n_init = warp_sum_u(n_init); n_ls = warp_sum_u(n_ls); n_fd = warp_sum_u(n_fd);
  if ((t & 31) == 0) {
    if (n_init) atomicAdd(&sh_ev[0], n_init);
    if (n_ls) atomicAdd(&sh_ev[1], n_ls);
    if (n_fd) atomicAdd(&sh_ev[2], n_fd);
  }
  __syncthreads();
  if (t == 0) {
    if (sh_ev[0]) atomicAdd(&s.ctrl->evals[EV_INIT], (unsigned long long)sh_ev[0]);
    if (sh_ev[1]) atomicAdd(&s.ctrl->evals[EV_LS], (unsigned long long)sh_ev[1]);
    if (sh_ev[2]) atomicAdd(&s.ctrl->evals[EV_LBFGS_FD], (unsigned long long)sh_ev[2]);
  }
}

inline size_t resident_extra_bytes() { return (size_t)2 * NT * 4; }

template <int OBJ, int DP>
cudaError_t launch_resident_dp(const DevObj &o, const ResArgs &a, int grid, size_t sh, cudaStream_t st) {
  if (a.s.m <= 8) k_lbfgs_resident<OBJ, DP, 8><<<grid, NT, sh, st>>>(o, a);
  else k_lbfgs_resident<OBJ, DP, 16><<<grid, NT, sh, st>>>(o, a);
  return cudaGetLastError();
}
template <int OBJ>
cudaError_t launch_resident_obj(const DevObj &o, const ResArgs &a, cudaStream_t st) {
  const int spt = NT / a.s.d, grid = (a.s.N + spt - 1) / spt;
  const size_t sh = eval_smem_bytes(o, resident_extra_bytes());
  if (o.DP == 8) return launch_resident_dp<OBJ, 8>(o, a, grid, sh, st);
  return launch_resident_dp<OBJ, 32>(o, a, grid, sh, st);
}
template <int OBJ>
cudaError_t configure_resident_obj() {
  cudaError_t e;
  const int big = 200 * 1024;
#define CHISAO_CFG_RES(DP_, MM_) \
  if ((e = cudaFuncSetAttribute(k_lbfgs_resident<OBJ, DP_, MM_>, cudaFuncAttributeMaxDynamicSharedMemorySize, big)) != cudaSuccess) return e;
  CHISAO_CFG_RES(8, 8) CHISAO_CFG_RES(8, 16) CHISAO_CFG_RES(32, 8) CHISAO_CFG_RES(32, 16)
#undef CHISAO_CFG_RES
  return cudaSuccess;
}

#define CHISAO_DECL_RES(ID) \
  cudaError_t launch_resident_obj_##ID(const DevObj &, const ResArgs &, cudaStream_t); \
  cudaError_t configure_resident_obj_##ID();
CHISAO_DECL_RES(0) CHISAO_DECL_RES(1) CHISAO_DECL_RES(2) CHISAO_DECL_RES(3) CHISAO_DECL_RES(4) CHISAO_DECL_RES(5)

}  // namespace chisao
