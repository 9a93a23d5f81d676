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

// ---- half-warp helpers: 16 lanes own one sample, lane hl holds coordinates 4 hl .. 4 hl + 3 ------------------
struct Row4 { float a, b, c, e; };
__device__ __forceinline__ Row4 ld_row4h(const float *row, int hl, int d, bool vec) {
  Row4 r;
  const int j = 4 * hl;
  if (vec) {
    if (j < d) { const float4 v = *reinterpret_cast<const float4 *>(row + j); r.a = v.x; r.b = v.y; r.c = v.z; r.e = v.w; }
    else { r.a = r.b = r.c = r.e = 0.f; }
  } else {
    r.a = (j < d) ? row[j] : 0.f; r.b = (j + 1 < d) ? row[j + 1] : 0.f;
    r.c = (j + 2 < d) ? row[j + 2] : 0.f; r.e = (j + 3 < d) ? row[j + 3] : 0.f;
  }
  return r;
}
__device__ __forceinline__ void st_row4h(float *row, int hl, int d, bool vec, Row4 r) {
  const int j = 4 * hl;
  if (vec) {
    if (j < d) *reinterpret_cast<float4 *>(row + j) = make_float4(r.a, r.b, r.c, r.e);
  } else {
    if (j < d) row[j] = r.a;
    if (j + 1 < d) row[j + 1] = r.b;
    if (j + 2 < d) row[j + 2] = r.c;
    if (j + 3 < d) row[j + 3] = r.e;
  }
}
__device__ __forceinline__ float half_sum(float v) {   // sum over the 16 lanes of a half-warp (all 32 lanes call)
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float half_max(float v) {
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float dot4(Row4 u, Row4 v) {
  return half_sum(fmaf(u.a, v.a, fmaf(u.b, v.b, fmaf(u.c, v.c, u.e * v.e))));
}
__device__ __forceinline__ void axpy4(Row4 &r, float c, Row4 v) {
  r.a = fmaf(c, v.a, r.a); r.b = fmaf(c, v.b, r.b); r.c = fmaf(c, v.c, r.c); r.e = fmaf(c, v.e, r.e);
}

// ---- history / state update after the FD gradient gn at the accepted trial point (R-4 (v), (vi)) ------------------
// Curvature pair s = x_t - x, y = gamma+ - gamma = g - gn, stored iff s.y > 1e-10 |s||y| (ring buffer, oldest dropped
// beyond m); x, f, g <- x_t, f(x_t), gn.  No trial accepted: stalled if the history was already empty, else the
// history is cleared.  Half-warp per sample; every lane of the warp calls (the dots are shuffles), `in` = the sample
// exists.  Returns the sample's state AFTER the update in registers, so that the two-loop recursion of the next
// iteration can follow in the same kernel (k_lbfgs_step).
struct SampleState { Row4 g, x; int len, head, stalled; bool have_x; unsigned bytes; };
template <bool VEC>
__device__ __forceinline__ SampleState lbfgs_update_half(const State &s, int i, bool in, int hl) {
  constexpr bool vec = VEC;
  const int d = s.d, m = s.m, N = s.N;
  const size_t ro = (size_t)(in ? i : 0) * d;
  SampleState o;
  const int b = in ? s.ls_b[i] : -2;
  o.len = in ? s.hist_len[i] : 0; o.head = in ? s.hist_head[i] : 0; o.stalled = in ? (int)s.stalled[i] : 0;
  o.g = ld_row4h(s.g + ro, hl, d, vec);
  if (!in) { o.g.a = o.g.b = o.g.c = o.g.e = 0.f; }
  o.x.a = o.x.b = o.x.c = o.x.e = 0.f; o.have_x = false; o.bytes = 0u;
  const bool acc = b >= 0;
  Row4 x = o.x, xt = o.x, gn = o.x;
  if (acc) { x = ld_row4h(s.x + ro, hl, d, vec); xt = ld_row4h(s.xt + ro, hl, d, vec); gn = ld_row4h(s.gn + ro, hl, d, vec); }
  Row4 sv, yv;
  sv.a = xt.a - x.a; sv.b = xt.b - x.b; sv.c = xt.c - x.c; sv.e = xt.e - x.e;
  yv.a = o.g.a - gn.a; yv.b = o.g.b - gn.b; yv.c = o.g.c - gn.c; yv.e = o.g.e - gn.e;
  const float sy = dot4(sv, yv), ss = dot4(sv, sv), yy = dot4(yv, yv);   // executed by all 32 lanes
  if (acc) {
    const float thr = 1e-10f * sqrtf(ss) * sqrtf(yy);
    o.bytes = 5u * d * 4u;                                 // x_t, gn, x read; x, g written
    if (sy > thr) {
      int ph;
      if (o.len == m) { ph = o.head; o.head = (o.head + 1 == m) ? 0 : o.head + 1; }
      else { ph = o.head + o.len; if (ph >= m) ph -= m; o.len += 1; }
      const size_t off = ((size_t)ph * s.hplane + (size_t)i * d);
      st_row4h(s.S + off, hl, d, vec, sv);
      st_row4h(s.Y + off, hl, d, vec, yv);
      if (hl == 0) { s.hist_len[i] = o.len; s.hist_head[i] = o.head; }
      o.bytes += 2u * d * 4u;
    }
    st_row4h(s.x + ro, hl, d, vec, xt);
    st_row4h(s.g + ro, hl, d, vec, gn);
    if (hl == 0) s.f[i] = s.ft[i];
    o.g = gn; o.x = xt; o.have_x = true;
  } else if (b == -1) {
    if (o.len == 0) { o.stalled = 1; if (hl == 0) s.stalled[i] = 1; }
    else { o.len = 0; o.head = 0; if (hl == 0) { s.hist_len[i] = 0; s.hist_head[i] = 0; } }
  }
  return o;
}

// One L-BFGS iteration, part 1: skip test, direction by the two-loop recursion (Nocedal & Wright Alg. 7.4;
// refs [19,20] of PAPER.md:77) with H0 = (s.y / y.y) I of the newest pair, steepest restart when the
// direction is not an ascent direction for f, first trial step and trial point (R-4).
// A half-warp owns one sample (two samples per warp, float4 per lane: one 512-byte contiguous request per warp
// and history plane); MM = compile-time bound on the history length, so the pair loops unroll over registers.
// Every shuffle is executed by all 32 lanes: inactive samples run with len = 0 and predicated stores.
// MODE: STEP_ALONE   the unit chisao_phase runs (state as stored);
//       STEP_FIRST   first iteration of a cycle: "stuck <- False^N" (Alg. 1) and the history reset of
//                    every Phase 1 (R-5) happen here instead of in a launch of their own;
//       STEP_UPDATE  iteration it >= 2 of a cycle: the update of iteration it - 1 (lbfgs_update_half) runs first, in the
//                    same kernel: one launch and one pass over x, g per iteration instead of two.
enum { STEP_ALONE = 0, STEP_FIRST = 1, STEP_UPDATE = 2 };
constexpr int DIR_WARPS = 4;   // measured at C5, full history: 4 warps x 4 CTAs per SM 4023 GB/s, 2 x 8 4025, 8 x 2 3884 (finer CTA turnover: less lockstep between load and recursion phases)
// SH: the 2 len history rows of a sample are staged in SHARED memory by cp.async (16 bytes per lane and row, no
// register staging) instead of being held in registers: 61 registers instead of 128 and five CTAs per SM instead of
// four.  Each lane reads back exactly the 16-byte chunks it copied, so no barrier is needed.  Needs d % 4 == 0 (VEC).
// Measured (B200, round 2): with short histories and many stationary samples -- the iterations of a cycle before the
// ring is full -- it is the faster form (C5 cycle: 0.62 against 0.78 ms for the 18 launches); with every sample active and
// a full ring the register form streams better (0.59 against 0.55 of the HBM copy bandwidth: the staged rows cost a
// shared-memory read in front of every shuffle-reduced dot, and the recursion's ~8 k cycles of dependent shuffles per
// sample, not the bytes in flight, bound both).  launch_lbfgs_step therefore stages through shared memory while the
// history cannot be full yet (iteration it <= m of a cycle) and keeps the rows in registers otherwise; a per-row
// bulk-copy (TMA) staging was measured too: 0.53.
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
template <int MM, bool VEC, int MODE, bool SH>
__global__ void __launch_bounds__(DIR_WARPS * 32, SH ? 5 : 4) k_lbfgs_step(State s, Hyper h) {
  extern __shared__ float4 hist_smem[];
  __shared__ int sh_cnt, sh_base;
  __shared__ unsigned int sh_bytes;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, hl = lane & 15, half = lane >> 4;
  const int i = (blockIdx.x * DIR_WARPS + wib) * 2 + half;
  const int d = s.d, m = s.m, N = s.N;
  constexpr bool vec = VEC;
  if (threadIdx.x == 0) { sh_cnt = 0; sh_bytes = 0u; }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    s.ctrl->ls_cnt[1] = 0; s.ctrl->ls_cnt[2] = 0; s.ctrl->fd_cnt = 0;
    if (MODE != STEP_ALONE) s.ctrl->fmax_enc = 0u;       // the cycle's f_max is accumulated by the last update of the pass
  }
  __syncthreads();
  const bool in = i < N;
  const size_t ro = (size_t)(in ? i : 0) * d;
  Row4 g, x;
  x.a = x.b = x.c = x.e = 0.f;
  int stalled_i, len_i, head_i;
  bool have_x = false;
  unsigned upd_bytes = 0u;
  if constexpr (MODE == STEP_UPDATE) {
    const SampleState u = lbfgs_update_half<VEC>(s, i, in, hl);
    g = u.g; x = u.x; have_x = u.have_x; stalled_i = u.stalled; len_i = u.len; head_i = u.head; upd_bytes = u.bytes;
  } else {
    // one round trip for everything the activity test needs (the flags are read whether or not the sample turns out
    // to be active: three dependent round trips -> two)
    g = ld_row4h(s.g + ro, hl, d, vec);
    if constexpr (MODE == STEP_FIRST) {
      stalled_i = 0; len_i = 0; head_i = 0;
      if (in && hl == 0) { s.stuck[i] = 0; s.removed[i] = 0; s.stalled[i] = 0; s.hist_len[i] = 0; s.hist_head[i] = 0; }
    } else {
      stalled_i = s.stalled[in ? i : 0]; len_i = s.hist_len[in ? i : 0]; head_i = s.hist_head[in ? i : 0];
    }
    if (!in) { g.a = g.b = g.c = g.e = 0.f; }
  }
  const float ginf = half_max(fmaxf(fmaxf(fabsf(g.a), fabsf(g.b)), fmaxf(fabsf(g.c), fabsf(g.e))));
  // (i) stationary (Eq. 3's gradient test) or stalled: no work, no evaluations (R-6)
  const bool act = in && !(stalled_i || !(ginf >= h.eps_grad));
  int len = act ? len_i : 0;
  const int len_read = len;
  const int head = act ? head_i : 0;
  Row4 Sr[SH ? 1 : MM], Yr[SH ? 1 : MM];
  float4 *hS = hist_smem + (size_t)((wib * 2 + half) * 2 * MM) * 16 + hl, *hY = hS + MM * 16;   // row l at [l * 16]
  // rows up to the longer history of the warp's two samples take part in the (warp-uniform) loops; the shorter
  // sample's missing rows are zero
  const int lw = SH ? max(len, __shfl_xor_sync(0xffffffffu, len, 16)) : MM;
  if constexpr (SH) {
    static_assert(!SH || VEC, "the shared-memory form needs float4 rows");
#pragma unroll
    for (int l = 0; l < MM; ++l) {
      if (l < len && 4 * hl < d) {
        int ph = head + l; if (ph >= m) ph -= m;
        const size_t off = ((size_t)ph * s.hplane + (size_t)i * d) + 4 * hl;
        cp_async16(hS + l * 16, s.S + off);
        cp_async16(hY + l * 16, s.Y + off);
      } else if (l < lw) {
        hS[l * 16] = make_float4(0.f, 0.f, 0.f, 0.f); hY[l * 16] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  } else {
#pragma unroll
  for (int l = 0; l < MM; ++l) {
    if (l < len) {
      int ph = head + l; if (ph >= m) ph -= m;
      const size_t off = ((size_t)ph * s.hplane + (size_t)i * d);
      Sr[l] = ld_row4h(s.S + off, hl, d, vec);
      Yr[l] = ld_row4h(s.Y + off, hl, d, vec);
    } else {
      Sr[l].a = Sr[l].b = Sr[l].c = Sr[l].e = 0.f; Yr[l] = Sr[l];
    }
  }
  }
  auto rowS = [&](int l) -> Row4 { if constexpr (SH) { const float4 v = hS[l * 16]; Row4 r; r.a = v.x; r.b = v.y; r.c = v.z; r.e = v.w; return r; } else return Sr[l]; };
  auto rowY = [&](int l) -> Row4 { if constexpr (SH) { const float4 v = hY[l * 16]; Row4 r; r.a = v.x; r.b = v.y; r.c = v.z; r.e = v.w; return r; } else return Yr[l]; };
  if (act && !have_x) x = ld_row4h(s.x + ro, hl, d, vec);
  // block-aggregated append of the searching samples to line-search worklist 0, and the byte counter: the one
  // returning global atomic per CTA is issued here, under the history loads, not at the end of the CTA's life
  int my_slot = 0;
  if (act && hl == 0) my_slot = atomicAdd(&sh_cnt, 1);
  if (in && hl == 0) atomicAdd(&sh_bytes, upd_bytes + (2u * d + (act ? 2u * (unsigned)len_read * d + 2u * d : 0u)) * 4u);
  __syncthreads();
  if (threadIdx.x == 0) {
    if (sh_cnt > 0) sh_base = atomicAdd(&s.ctrl->ls_cnt[0], sh_cnt);
    if (sh_bytes) atomicAdd(&s.ctrl->evals[7], (unsigned long long)sh_bytes);   // g read, p written (+ pairs, x, x_t; + the update's rows)
  }
  Row4 gam; gam.a = -g.a; gam.b = -g.b; gam.c = -g.c; gam.e = -g.e;
  // a warp none of whose two samples is active skips the recursion altogether (late in phase 2 most are stationary)
  Row4 p, xt;
  p.a = p.b = p.c = p.e = 0.f; xt = p;
  bool restart = false;
  float t0 = 0.f, dec = 0.f;
  if constexpr (SH) asm volatile("cp.async.wait_all;" ::: "memory");
  if (__any_sync(0xffffffffu, act)) {
  const float gn2 = dot4(g, g);
  // straight-line code over all MM slots: rows beyond len are zero and rho = 0 there, so they contribute nothing,
  // and no shuffle sits under a branch (the compiler would otherwise wrap each one in a convergence region)
  float rho[MM], al[MM];
#pragma unroll
  for (int l = 0; l < MM; ++l) {
    rho[l] = 0.0f; al[l] = 0.0f;
    if (l < lw) { const float sy = dot4(rowS(l), rowY(l)); rho[l] = (l < len) ? 1.0f / sy : 0.0f; }
  }
  Row4 r = gam;
  // (shared-memory form: the rows of step l - 1 are fetched before the shuffle chain of step l starts)
  Row4 Sn = rowS(SH ? max(lw - 1, 0) : MM - 1), Ynx = rowY(SH ? max(lw - 1, 0) : MM - 1);
#pragma unroll
  for (int l = MM - 1; l >= 0; --l) if (l < lw) {
    const Row4 Sc = SH ? Sn : rowS(l), Yc = SH ? Ynx : rowY(l);
    if (SH && l > 0) { Sn = rowS(l - 1); Ynx = rowY(l - 1); }
    al[l] = rho[l] * dot4(Sc, r); axpy4(r, -al[l], Yc);
  }
  // newest pair (logical len - 1): its y row is re-read (an L1/L2 hit) rather than selected out of the register
  // array, which would turn the array into local memory; s.y of that pair = 1 / rho
  Row4 Yn; Yn.a = Yn.b = Yn.c = Yn.e = 0.f;
  float rho_n = 1.0f;
  if (len > 0) {
    if constexpr (SH) Yn = rowY(len - 1);                // (shared memory can be indexed dynamically)
    else {
      int ph = head + len - 1; if (ph >= m) ph -= m;
      Yn = ld_row4h(s.Y + ((size_t)ph * s.hplane + (size_t)i * d), hl, d, vec);
    }
  }
#pragma unroll
  for (int l = 0; l < MM; ++l) rho_n = (l == len - 1) ? rho[l] : rho_n;
  if (len > 0) { const float h0 = 1.0f / (rho_n * dot4(Yn, Yn)); r.a *= h0; r.b *= h0; r.c *= h0; r.e *= h0; }
  else { (void)dot4(Yn, Yn); }
#pragma unroll
  Sn = rowS(0); Ynx = rowY(0);
#pragma unroll
  for (int l = 0; l < MM; ++l) if (l < lw) {
    const Row4 Sc = SH ? Sn : rowS(l), Yc = SH ? Ynx : rowY(l);
    if (SH && l + 1 < lw) { Sn = rowS(l + 1); Ynx = rowY(l + 1); }
    const float beta = rho[l] * dot4(Yc, r); axpy4(r, al[l] - beta, Sc);
  }
  p.a = -r.a; p.b = -r.b; p.c = -r.c; p.e = -r.e;
  const float gp = dot4(gam, p);
  restart = false;
  if (len > 0 && !(gp < 0.0f)) { restart = true; len = 0; }   // not a descent direction for phi = -f: steepest restart
  if (len_read == 0 || restart) { p.a = -gam.a; p.b = -gam.b; p.c = -gam.c; p.e = -gam.e; }
  // (iii) first trial step; (iv) trial point projected on Theta, Armijo linear term gamma.(x_t - x)
  t0 = (len > 0) ? 1.0f : fminf(1.0f, 1.0f / sqrtf(gn2));
  const Row4 lo = ld_row4h(s.lo, hl, d, vec), hi = ld_row4h(s.hi, hl, d, vec);
  xt.a = clipf(fmaf(t0, p.a, x.a), lo.a, hi.a); xt.b = clipf(fmaf(t0, p.b, x.b), lo.b, hi.b);
  xt.c = clipf(fmaf(t0, p.c, x.c), lo.c, hi.c); xt.e = clipf(fmaf(t0, p.e, x.e), lo.e, hi.e);
  Row4 dx; dx.a = xt.a - x.a; dx.b = xt.b - x.b; dx.c = xt.c - x.c; dx.e = xt.e - x.e;
  dec = dot4(gam, dx);
  }
  if (in) {
    if (act) {
      st_row4h(s.xt + ro, hl, d, vec, xt);
      st_row4h(s.p + ro, hl, d, vec, p);
      if (hl == 0) {
        s.dec[i] = dec; s.tcur[i] = t0; s.ls_b[i] = -1;
        if (restart) { s.hist_len[i] = 0; s.hist_head[i] = 0; }
      }
    } else {
      Row4 z; z.a = z.b = z.c = z.e = 0.f;
      st_row4h(s.p + ro, hl, d, vec, z);
      if (hl == 0) s.ls_b[i] = -2;
    }
  }
  __syncthreads();                     // sh_base (written by thread 0 after its atomic returned)
  if (act && hl == 0) s.ls_list[0][sh_base + my_slot] = i;
}

// One L-BFGS iteration, part 3 as a launch of its own (the unit chisao_phase runs, and the last iteration of a pass):
// lbfgs_update_half for every sample.  STICK: also Phase 2's per-sample ||grad f||_inf and the f_max partials (what
// k_ginf_fmax computes, chisao_select.cu), from the gradient and value this kernel has just written -- at the end of
// a pass the stick test follows at once.
template <bool VEC, bool STICK>
__global__ void __launch_bounds__(DIR_WARPS * 32) k_lbfgs_update(State s, Hyper h) {
  __shared__ float sh_max[DIR_WARPS];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, hl = lane & 15, half = lane >> 4;
  const int i = (blockIdx.x * DIR_WARPS + wib) * 2 + half;
  if (blockIdx.x == 0 && threadIdx.x == 0) s.ctrl->ls_cnt[0] = 0;
  const bool in = i < s.N;
  const SampleState u = lbfgs_update_half<VEC>(s, i, in, hl);
  if constexpr (STICK) {
    const float a0 = fabsf(u.g.a), a1 = fabsf(u.g.b), a2 = fabsf(u.g.c), a3 = fabsf(u.g.e);
    const bool nan = !(a0 == a0) || !(a1 == a1) || !(a2 == a2) || !(a3 == a3);
    const float gi = half_max(fmaxf(fmaxf(a0, a1), fmaxf(a2, a3)));
    const unsigned nanmask = __ballot_sync(0xffffffffu, nan);
    const bool any_nan = (nanmask >> (16 * half)) & 0xFFFFu;
    float fm = -INFINITY;
    if (in && hl == 0) {
      s.ginf[i] = any_nan ? NAN : gi;                    // a NaN gradient can never pass "< eps_grad"
      const float f = s.f[i];                            // written above by this lane if the trial was accepted
      if (fabsf(f) <= 3.0e38f) fm = f;                   // finite values only (R-13)
    }
    fm = warp_max(fm);
    if (lane == 0) sh_max[wib] = fm;
    __syncthreads();
    if (threadIdx.x == 0) {
      float mx = sh_max[0];
#pragma unroll
      for (int w = 1; w < DIR_WARPS; ++w) mx = fmaxf(mx, sh_max[w]);
      if (mx > -INFINITY) atomicMax(&s.ctrl->fmax_enc, enc_ordered(mx));
    }
  }
  if (in && hl == 0 && u.bytes) atomicAdd(&s.ctrl->evals[7], (unsigned long long)u.bytes);
}

cudaError_t launch_release(const State &s, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  k_release<<<(s.N + 255) / 256, 256, 0, st>>>(s);
  return cudaGetLastError();
}
static bool g_step_regs = false;   // CHISAO_STEP_REGS in the environment: keep the register form of the history (A/B measurements)
template <int MM, bool VEC, int MODE, bool SH>
static cudaError_t launch_step_one(const State &s, const Hyper &h, int grid, cudaStream_t st) {
  const size_t sh = SH ? (size_t)DIR_WARPS * 2 * 2 * MM * 16 * sizeof(float4) : 0;
  if (SH) {
    static bool configured = false;
    if (!configured) {
      cudaError_t e = cudaFuncSetAttribute(k_lbfgs_step<MM, VEC, MODE, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
      if (e != cudaSuccess) return e;
      configured = true;
    }
  }
  k_lbfgs_step<MM, VEC, MODE, SH><<<grid, DIR_WARPS * 32, sh, st>>>(s, h);
  return cudaGetLastError();
}
template <int MM, bool VEC, bool SH>
static cudaError_t launch_step_mode(const State &s, const Hyper &h, int mode, int grid, cudaStream_t st) {
  if (mode == STEP_FIRST) return launch_step_one<MM, VEC, STEP_FIRST, false>(s, h, grid, st);   // (empty history: nothing to stage)
  if (mode == STEP_UPDATE) return launch_step_one<MM, VEC, STEP_UPDATE, SH>(s, h, grid, st);
  return launch_step_one<MM, VEC, STEP_ALONE, SH>(s, h, grid, st);
}
template <int MM>
static cudaError_t launch_step_mm(const State &s, const Hyper &h, int mode, bool staged, int grid, cudaStream_t st) {
  const bool vec = (s.d & 3) == 0;
  if (!vec) return launch_step_mode<MM, false, false>(s, h, mode, grid, st);
  if (!staged) return launch_step_mode<MM, true, false>(s, h, mode, grid, st);
  return launch_step_mode<MM, true, true>(s, h, mode, grid, st);
}
// `it`: iteration of the cycle (0 for the stand-alone unit): after it - 1 updates a history holds at most it - 1 pairs
cudaError_t launch_lbfgs_step(const State &s, const Hyper &h, int mode, int it, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  static bool env_read = false;
  if (!env_read) { g_step_regs = getenv("CHISAO_STEP_REGS") != nullptr; env_read = true; }
  const int per_block = DIR_WARPS * 2, grid = (s.N + per_block - 1) / per_block;
  const bool staged = !g_step_regs && mode == STEP_UPDATE && it - 1 < s.m;   // the ring cannot be full yet
  if (s.m <= 4) return launch_step_mm<4>(s, h, mode, staged, grid, st);
  if (s.m <= 8) return launch_step_mm<8>(s, h, mode, staged, grid, st);
  if (s.m <= 10) return launch_step_mm<10>(s, h, mode, staged, grid, st);
  return launch_step_mm<16>(s, h, mode, staged, grid, st);
}
cudaError_t launch_lbfgs_update(const State &s, const Hyper &h, bool stick_partials, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  const int per_block = DIR_WARPS * 2, grid = (s.N + per_block - 1) / per_block;
  const bool vec = (s.d & 3) == 0;
  if (vec) {
    if (stick_partials) k_lbfgs_update<true, true><<<grid, DIR_WARPS * 32, 0, st>>>(s, h);
    else k_lbfgs_update<true, false><<<grid, DIR_WARPS * 32, 0, st>>>(s, h);
  } else {
    if (stick_partials) k_lbfgs_update<false, true><<<grid, DIR_WARPS * 32, 0, st>>>(s, h);
    else k_lbfgs_update<false, false><<<grid, DIR_WARPS * 32, 0, st>>>(s, h);
  }
  return cudaGetLastError();
}

}  // namespace chisao
