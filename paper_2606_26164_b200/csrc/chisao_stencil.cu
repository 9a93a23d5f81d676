// chisao_stencil.cu -- stencil-aware FD evaluator for the dense objectives (
// PAPER.md:555 names the 2dN finite-difference evaluations as the cost lever).  OPT-IN (phase_mask bit
// CHISAO_FLAG_STENCIL_AWARE) and reported separately from the black-box numbers: it uses the structure of the
// objective, which a value-only oracle f(theta) does not expose.
//
// For q_k(x) = || W_k (x - mu_k) ||^2 the 2d stencil points x +- delta e_j share the base quantities of the centre:
//     z = W_k (x - mu_k),  q0 = |z|^2,  t = W_k^T z,  cc_j = sum_n W_k[n][j]^2
//     q_k(x +- delta e_j) = q0 +- 2 delta t_j + delta^2 cc_j                      (exact identity)
// so one component costs two d x d matrix-vector products per SAMPLE instead of one per stencil POINT (2d of them):
// d times less arithmetic.  The 2d values f(x +- delta e_j) = lse_k (a_k - q_k/2) (QUAD: -q/2) are the same
// quantities the black-box path computes, within rounding; noise draws, the fp32 step actually taken, the gradient
// formula and the Eq. 6 epilogue are those of k_eval_fd (chisao_eval_kernels.cuh).
//
// Mapping: one thread per sample, 128 samples per CTA.  x sits in shared memory as float4 columns (thread-private
// column, conflict-free); d = x - mu and t live in registers; W_k rows are broadcast from the streamed record
// (cp.async.bulk + mbarrier, double-buffered); the 2d online log-sum-exp states (m, s) of a sample live in shared
// memory as [stencil point][thread] float2 (conflict-free).
#include "chisao_eval_kernels.cuh"

namespace chisao {

constexpr int ST_NT = 128;

template <int DP>
struct StencilSmem {
  static constexpr size_t rec_floats = (size_t)DP * DP + DP + 4;
  static constexpr size_t off_rec = 16;                                            // two mbarriers first
  static constexpr size_t off_cc = off_rec + 2 * rec_floats * 4;                   // cc[DP]
  static constexpr size_t off_x = off_cc + DP * 4;                                 // x as float4 [DP/4][ST_NT]
  static constexpr size_t off_st = off_x + (size_t)(DP / 4) * ST_NT * 16;          // float2 [2 DP][ST_NT]
  static constexpr size_t bytes_quad = off_st;
  static constexpr size_t bytes_gmm = off_st + (size_t)2 * DP * ST_NT * 8;
};

template <int OBJ, int DP>
__global__ void __launch_bounds__(ST_NT, 1) k_fd_stencil(const DevObj o, const FdArgs a) {
  using L = StencilSmem<DP>;
  extern __shared__ __align__(16) unsigned char st_smem[];
  uint64_t *bar = reinterpret_cast<uint64_t *>(st_smem);
  float *recbuf = reinterpret_cast<float *>(st_smem + L::off_rec);
  float *cc = reinterpret_cast<float *>(st_smem + L::off_cc);
  float4 *xs = reinterpret_cast<float4 *>(st_smem + L::off_x);
  float2 *stt = reinterpret_cast<float2 *>(st_smem + L::off_st);
  const int t = threadIdx.x, d = a.d;
  const int cnt = a.count ? *a.count : a.max_count;
  const int first = blockIdx.x * ST_NT;
  if (blockIdx.x == 0 && t == 0 && a.zero_cnt) *a.zero_cnt = 0;
  if (first >= cnt) return;
  if (t == 0) { mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_fence_init(); }
  const bool valid = first + t < cnt;
  const int i = valid ? (a.list ? a.list[first + t] : first + t) : 0;
  const bool vec = (d & 3) == 0;
  const float *row = a.X + (size_t)i * d;
#pragma unroll
  for (int c4 = 0; c4 < DP / 4; ++c4)
    xs[c4 * ST_NT + t] = valid ? ld_row4(row, c4, d, vec) : make_float4(0.f, 0.f, 0.f, 0.f);
  if constexpr (OBJ == CHISAO_OBJ_GMM_FULL) {
#pragma unroll 4
    for (int p = 0; p < 2 * DP; ++p) stt[p * ST_NT + t] = make_float2(-INFINITY, 0.0f);
  }
  __syncthreads();                                     // barriers initialised
  const uint32_t rec_bytes = (uint32_t)L::rec_floats * 4;
  if (t == 0) { mbar_expect_tx(&bar[0], rec_bytes); bulk_g2s(recbuf, o.recs, rec_bytes, &bar[0]); }
  const float *xf = reinterpret_cast<const float *>(xs);   // coordinate c of this thread: xf[((c >> 2) * ST_NT + t) * 4 + (c & 3)]
  float qsum = 0.0f;                                   // QUAD keeps q0 and t of its single component
  float tq[DP];
  for (int k = 0; k < o.K; ++k) {
    const int b = k & 1;
    if (k + 1 < o.K && t == 0) {                       // buffer b ^ 1 was released by the barrier ending iteration k - 1
      mbar_expect_tx(&bar[b ^ 1], rec_bytes);
      bulk_g2s(recbuf + (size_t)(b ^ 1) * L::rec_floats, o.recs + (size_t)(k + 1) * L::rec_floats, rec_bytes, &bar[b ^ 1]);
    }
    mbar_wait(&bar[b], (k >> 1) & 1);
    const float *W = recbuf + (size_t)b * L::rec_floats;
    const float4 *mu4 = reinterpret_cast<const float4 *>(W + DP * DP);
    const float a_k = W[DP * DP + DP];
    if (t < DP) {                                      // cc_j = sum_n W[n][j]^2 (lanes read consecutive addresses)
      float acc = 0.0f;
#pragma unroll 8
      for (int n = 0; n < DP; ++n) { const float w = W[n * DP + t]; acc = fmaf(w, w, acc); }
      cc[t] = acc;
    }
    float df[DP], tt[DP];
#pragma unroll
    for (int c4 = 0; c4 < DP / 4; ++c4) {
      const float4 v = xs[c4 * ST_NT + t], m = mu4[c4];
      df[4 * c4] = v.x - m.x; df[4 * c4 + 1] = v.y - m.y; df[4 * c4 + 2] = v.z - m.z; df[4 * c4 + 3] = v.w - m.w;
      tt[4 * c4] = 0.f; tt[4 * c4 + 1] = 0.f; tt[4 * c4 + 2] = 0.f; tt[4 * c4 + 3] = 0.f;
    }
    float q0 = 0.0f;
#pragma unroll 2
    for (int n = 0; n < DP; ++n) {
      const float4 *W4 = reinterpret_cast<const float4 *>(W + n * DP);
      float4 w[DP / 4];
      float z0 = 0.f, z1 = 0.f, z2 = 0.f, z3 = 0.f;
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        w[c4] = W4[c4];
        z0 = fmaf(w[c4].x, df[4 * c4], z0); z1 = fmaf(w[c4].y, df[4 * c4 + 1], z1);
        z2 = fmaf(w[c4].z, df[4 * c4 + 2], z2); z3 = fmaf(w[c4].w, df[4 * c4 + 3], z3);
      }
      const float z = (z0 + z1) + (z2 + z3);
      q0 = fmaf(z, z, q0);
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        tt[4 * c4] = fmaf(w[c4].x, z, tt[4 * c4]); tt[4 * c4 + 1] = fmaf(w[c4].y, z, tt[4 * c4 + 1]);
        tt[4 * c4 + 2] = fmaf(w[c4].z, z, tt[4 * c4 + 2]); tt[4 * c4 + 3] = fmaf(w[c4].w, z, tt[4 * c4 + 3]);
      }
    }
    __syncthreads();                                   // cc visible
    if constexpr (OBJ == CHISAO_OBJ_QUAD) {
      qsum = q0;
#pragma unroll
      for (int c = 0; c < DP; ++c) tq[c] = tt[c];
    } else {
#pragma unroll
      for (int j = 0; j < DP; ++j) {
        if (j < d) {
          const float xj = xf[((j >> 2) * ST_NT + t) * 4 + (j & 3)];
          const float dp = (xj + a.h) - xj, dm = xj - (xj - a.h);       // the steps actually taken in fp32 (R-1)
          const float ccj = cc[j];
          const float qp = fmaf(dp, fmaf(dp, ccj, 2.0f * tt[j]), q0);   // q0 + 2 dp t_j + dp^2 cc_j
          const float qm = fmaf(dm, fmaf(dm, ccj, -2.0f * tt[j]), q0);  // q0 - 2 dm t_j + dm^2 cc_j
          {
            float2 s = stt[(2 * j) * ST_NT + t];
            const float v = fmaf(-0.5f, qp, a_k), mn = fmaxf(s.x, v);
            if (mn > -INFINITY) { s.y = s.y * __expf(s.x - mn) + __expf(v - mn); s.x = mn; }
            stt[(2 * j) * ST_NT + t] = s;
          }
          {
            float2 s = stt[(2 * j + 1) * ST_NT + t];
            const float v = fmaf(-0.5f, qm, a_k), mn = fmaxf(s.x, v);
            if (mn > -INFINITY) { s.y = s.y * __expf(s.x - mn) + __expf(v - mn); s.x = mn; }
            stt[(2 * j + 1) * ST_NT + t] = s;
          }
        }
      }
    }
    __syncthreads();                                   // record buffer b and cc are free again
  }
  if (valid) {
#pragma unroll
    for (int j = 0; j < DP; ++j) {
      if (j < d) {
        const float xj = xf[((j >> 2) * ST_NT + t) * 4 + (j & 3)];
        const float xph = xj + a.h, xmh = xj - a.h;
        float fp, fm;
        if constexpr (OBJ == CHISAO_OBJ_QUAD) {
          const float dp = xph - xj, dm = xj - xmh, ccj = cc[j];
          fp = -0.5f * fmaf(dp, fmaf(dp, ccj, 2.0f * tq[j]), qsum);
          fm = -0.5f * fmaf(dm, fmaf(dm, ccj, -2.0f * tq[j]), qsum);
        } else {
          const float2 sp = stt[(2 * j) * ST_NT + t], sm_ = stt[(2 * j + 1) * ST_NT + t];
          fp = sp.x + logf(sp.y); fm = sm_.x + logf(sm_.y);
        }
        fp += eval_noise(o.sigma_noise, a.seed, a.cycle, i, a.phase, a.iter, a.slot_off + 1 + 2 * j);
        fm += eval_noise(o.sigma_noise, a.seed, a.cycle, i, a.phase, a.iter, a.slot_off + 2 + 2 * j);
        const float g = (fp - fm) / ((xph - xj) + (xj - xmh));
        if (a.mode == FD_GRAD) {
          a.g_out[(size_t)i * d + j] = g;
        } else {  // Eq. 6
          const float vo = (a.iter == 1) ? 0.0f : a.v[(size_t)i * d + j];
          const float vn = fmaf(a.mu, vo, -a.alpha * g);
          a.v[(size_t)i * d + j] = vn;
          a.x[(size_t)i * d + j] = clipf(xj + vn, a.lo[j], a.hi[j]);
        }
      }
    }
  }
  if (t == 0) atomicAdd(&a.evals[a.counter], (unsigned long long)min(ST_NT, cnt - first) * 2ull * d);
}

template <int OBJ, int DP>
static cudaError_t launch_one(const DevObj &o, const FdArgs &a, int n_samples, cudaStream_t st) {
  using L = StencilSmem<DP>;
  const size_t sh = (OBJ == CHISAO_OBJ_QUAD) ? L::bytes_quad : L::bytes_gmm;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_fd_stencil<OBJ, DP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  k_fd_stencil<OBJ, DP><<<(n_samples + ST_NT - 1) / ST_NT, ST_NT, sh, st>>>(o, a);
  return cudaGetLastError();
}

bool fd_stencil_supported(const DevObj &o) { return o.id == CHISAO_OBJ_GMM_FULL || o.id == CHISAO_OBJ_QUAD; }

cudaError_t launch_fd_stencil(const DevObj &o, const FdArgs &a, int n_samples, cudaStream_t st) {
#define CHISAO_ST(OBJ)                                                     \
  switch (o.DP) {                                                          \
    case 8: return launch_one<OBJ, 8>(o, a, n_samples, st);                \
    case 32: return launch_one<OBJ, 32>(o, a, n_samples, st);              \
    default: return launch_one<OBJ, 64>(o, a, n_samples, st);              \
  }
  if (o.id == CHISAO_OBJ_QUAD) { CHISAO_ST(CHISAO_OBJ_QUAD) }
  CHISAO_ST(CHISAO_OBJ_GMM_FULL)
#undef CHISAO_ST
}

}  // namespace chisao
