// chisao_lbfgs.cu -- Phase 1 state kernels (Eq. 2): release, two-loop recursion over the
// (s, y) history spilled to HBM, first line-search trial point, and the history / state update after the
// finite-difference gradient at the accepted trial point.  Readings R-4, R-5, R-6.
//
// Layout: history S, Y are [m][N][d] ring buffers (physical slot planes); logical pair l (0 = oldest) of
// sample i lives in plane (head_i + l) mod m.  One warp owns one sample: lane L holds coordinates 2L and
// 2L+1 (float2, one fully coalesced 256-byte row per warp instruction at d = 64); all 2*len history rows
// are loaded into registers once and serve both loops of the recursion.  This kernel is HBM-bound
// ((2 len d + 6 d) * 4 bytes per sample-iteration).
#include "chisao_device.cuh"

namespace chisao {

constexpr int WARPS_PER_BLOCK = 8;

struct Row2 { float a, b; };
__device__ __forceinline__ Row2 ld_row2(const float *row, int lane, int d, bool even) {
  Row2 r;
  const int j = 2 * lane;
  if (even) {
    if (j < d) { const float2 v = *reinterpret_cast<const float2 *>(row + j); r.a = v.x; r.b = v.y; }
    else { r.a = 0.f; r.b = 0.f; }
  } else {
    r.a = (j < d) ? row[j] : 0.f;
    r.b = (j + 1 < d) ? row[j + 1] : 0.f;
  }
  return r;
}
__device__ __forceinline__ void st_row2(float *row, int lane, int d, bool even, Row2 r) {
  const int j = 2 * lane;
  if (even) {
    if (j < d) *reinterpret_cast<float2 *>(row + j) = make_float2(r.a, r.b);
  } else {
    if (j < d) row[j] = r.a;
    if (j + 1 < d) row[j + 1] = r.b;
  }
}
__device__ __forceinline__ float dot2(Row2 u, Row2 v) { return warp_sum(fmaf(u.a, v.a, u.b * v.b)); }

// "stuck <- False^N" (Alg. 1) + history reset at the start of every Phase 1 (R-5)
__global__ void k_release(State s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  s.stuck[i] = 0; s.removed[i] = 0; s.stalled[i] = 0; s.hist_len[i] = 0; s.hist_head[i] = 0;
}

// One L-BFGS iteration, part 1: skip test, direction by the two-loop recursion (Nocedal & Wright Alg. 7.4;
// refs [19,20] of PAPER.md:77) with H0 = (s.y / y.y) I of the newest pair, steepest restart when the
// direction is not an ascent direction for f, first trial step and trial point (R-4).
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) k_lbfgs_direction(State s, Hyper h) {
  __shared__ int sh_cnt, sh_base;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int i = blockIdx.x * WARPS_PER_BLOCK + wib;
  const int d = s.d, m = s.m, N = s.N;
  const bool even = (d & 1) == 0;
  if (threadIdx.x == 0) sh_cnt = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) { s.ctrl->ls_cnt[1] = 0; s.ctrl->ls_cnt[2] = 0; s.ctrl->fd_cnt = 0; }
  __syncthreads();
  bool search = false;
  int my_slot = 0;
  if (i < N) {
    const size_t ro = (size_t)i * d;
    const Row2 g = ld_row2(s.g + ro, lane, d, even);
    const float ginf = warp_max(fmaxf(fabsf(g.a), fabsf(g.b)));
    // (i) stationary (Eq. 3's gradient test) or stalled: no work, no evaluations (R-6)
    const bool skip = s.stalled[i] || !(ginf >= h.eps_grad);
    Row2 p; p.a = 0.f; p.b = 0.f;
    if (skip) {
      if (lane == 0) s.ls_b[i] = -2;
    } else {
      int len = s.hist_len[i];
      const int head = s.hist_head[i];
      const Row2 x = ld_row2(s.x + ro, lane, d, even);
      Row2 gam; gam.a = -g.a; gam.b = -g.b;
      const float gn2 = dot2(g, g);
      if (len > 0) {
        Row2 Sr[CHISAO_MAX_M], Yr[CHISAO_MAX_M];
#pragma unroll
        for (int l = 0; l < CHISAO_MAX_M; ++l) {
          if (l < len) {
            int ph = head + l; if (ph >= m) ph -= m;
            const size_t off = ((size_t)ph * N + i) * d;
            Sr[l] = ld_row2(s.S + off, lane, d, even);
            Yr[l] = ld_row2(s.Y + off, lane, d, even);
          }
        }
        float rho[CHISAO_MAX_M], al[CHISAO_MAX_M];
#pragma unroll
        for (int l = 0; l < CHISAO_MAX_M; ++l)
          if (l < len) rho[l] = 1.0f / dot2(Sr[l], Yr[l]);
        Row2 r = gam;
#pragma unroll
        for (int l = CHISAO_MAX_M - 1; l >= 0; --l) {
          if (l < len) {
            al[l] = rho[l] * dot2(Sr[l], r);
            r.a = fmaf(-al[l], Yr[l].a, r.a); r.b = fmaf(-al[l], Yr[l].b, r.b);
          }
        }
        float sy = 0.f, yy = 1.f;
#pragma unroll
        for (int l = 0; l < CHISAO_MAX_M; ++l)
          if (l == len - 1) { sy = dot2(Sr[l], Yr[l]); yy = dot2(Yr[l], Yr[l]); }
        const float h0 = sy / yy;
        r.a *= h0; r.b *= h0;
#pragma unroll
        for (int l = 0; l < CHISAO_MAX_M; ++l) {
          if (l < len) {
            const float beta = rho[l] * dot2(Yr[l], r);
            const float c = al[l] - beta;
            r.a = fmaf(Sr[l].a, c, r.a); r.b = fmaf(Sr[l].b, c, r.b);
          }
        }
        p.a = -r.a; p.b = -r.b;
        const float gp = dot2(gam, p);
        if (!(gp < 0.0f)) {  // not a descent direction for phi = -f: steepest restart, clear history
          p.a = -gam.a; p.b = -gam.b;
          len = 0;
          if (lane == 0) { s.hist_len[i] = 0; s.hist_head[i] = 0; }
        }
      } else {
        p.a = -gam.a; p.b = -gam.b;
      }
      // (iii) first trial step; (iv) trial point projected on Theta, Armijo linear term gamma.(x_t - x)
      const float t0 = (len > 0) ? 1.0f : fminf(1.0f, 1.0f / sqrtf(gn2));
      const Row2 lo = ld_row2(s.lo, lane, d, even), hi = ld_row2(s.hi, lane, d, even);
      Row2 xt;
      xt.a = clipf(fmaf(t0, p.a, x.a), lo.a, hi.a);
      xt.b = clipf(fmaf(t0, p.b, x.b), lo.b, hi.b);
      Row2 dx; dx.a = xt.a - x.a; dx.b = xt.b - x.b;
      const float dec = dot2(gam, dx);
      st_row2(s.xt + ro, lane, d, even, xt);
      if (lane == 0) { s.dec[i] = dec; s.tcur[i] = t0; s.ls_b[i] = -1; }
      search = true;
    }
    st_row2(s.p + ro, lane, d, even, p);
  }
  // block-aggregated append of the searching samples to line-search worklist 0
  if (search && lane == 0) my_slot = atomicAdd(&sh_cnt, 1);
  __syncthreads();
  if (threadIdx.x == 0 && sh_cnt > 0) sh_base = atomicAdd(&s.ctrl->ls_cnt[0], sh_cnt);
  __syncthreads();
  if (search && lane == 0) s.ls_list[0][sh_base + my_slot] = i;
}

// One L-BFGS iteration, part 3 (after the FD gradient gn at the accepted trial point): curvature pair
// s = x_t - x, y = gamma+ - gamma = g - gn, stored iff s.y > 1e-10 |s||y| (ring buffer, oldest dropped
// beyond m); x, f, g <- x_t, f(x_t), gn.  No trial accepted: stalled if the history was already empty,
// else the history is cleared (R-4 (v), (vi)).
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) k_lbfgs_update(State s, Hyper h) {
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int i = blockIdx.x * WARPS_PER_BLOCK + wib;
  if (blockIdx.x == 0 && threadIdx.x == 0) s.ctrl->ls_cnt[0] = 0;
  if (i >= s.N) return;
  const int d = s.d, m = s.m, N = s.N;
  const bool even = (d & 1) == 0;
  const int b = s.ls_b[i];
  if (b == -2) return;
  int len = s.hist_len[i], head = s.hist_head[i];
  if (b < 0) {
    if (lane == 0) {
      if (len == 0) s.stalled[i] = 1; else { s.hist_len[i] = 0; s.hist_head[i] = 0; }
    }
    return;
  }
  const size_t ro = (size_t)i * d;
  const Row2 x = ld_row2(s.x + ro, lane, d, even), xt = ld_row2(s.xt + ro, lane, d, even);
  const Row2 g = ld_row2(s.g + ro, lane, d, even), gn = ld_row2(s.gn + ro, lane, d, even);
  Row2 sv, yv;
  sv.a = xt.a - x.a; sv.b = xt.b - x.b;
  yv.a = g.a - gn.a; yv.b = g.b - gn.b;
  const float sy = dot2(sv, yv), ss = dot2(sv, sv), yy = dot2(yv, yv);
  const float thr = 1e-10f * sqrtf(ss) * sqrtf(yy);
  if (sy > thr) {
    int ph;
    if (len == m) { ph = head; head = (head + 1 == m) ? 0 : head + 1; }
    else { ph = head + len; if (ph >= m) ph -= m; len += 1; }
    const size_t off = ((size_t)ph * N + i) * d;
    st_row2(s.S + off, lane, d, even, sv);
    st_row2(s.Y + off, lane, d, even, yv);
    if (lane == 0) { s.hist_len[i] = len; s.hist_head[i] = head; }
  }
  st_row2(s.x + ro, lane, d, even, xt);
  st_row2(s.g + ro, lane, d, even, gn);
  if (lane == 0) s.f[i] = s.ft[i];
}

cudaError_t launch_release(const State &s, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  k_release<<<(s.N + 255) / 256, 256, 0, st>>>(s);
  return cudaGetLastError();
}
cudaError_t launch_lbfgs_direction(const State &s, const Hyper &h, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  k_lbfgs_direction<<<(s.N + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK, WARPS_PER_BLOCK * 32, 0, st>>>(s, h);
  return cudaGetLastError();
}
cudaError_t launch_lbfgs_update(const State &s, const Hyper &h, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  k_lbfgs_update<<<(s.N + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK, WARPS_PER_BLOCK * 32, 0, st>>>(s, h);
  return cudaGetLastError();
}

}  // namespace chisao
