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
  const int d = s.d, m = s.m;
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
__global__ void __launch_bounds__(DIR_WARPS * 32, SH ? 5 : 4) k_lbfgs_step(State s, Hyper h, int hrows) {
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
  // (hrows <= MM rows per sample and array are staged: inside a cycle a history holds at most it - 1 pairs, and the fewer
  // rows a CTA reserves the more CTAs an SM holds)
  float4 *hS = hist_smem + (size_t)((wib * 2 + half) * 2 * hrows) * 16 + hl, *hY = hS + hrows * 16;   // row l at [l * 16]
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

// ---- QUAD form of the step kernel: four lanes own one sample, the history planes of a warp's eight samples are
// bulk-copied (TMA engine, one 2 KB copy per plane at d = 64) into shared memory -----------------------------------------
// Why: with 16 lanes per sample a dot product is 4 FMAs and 4 dependent shuffle steps, and a warp instruction covers two
// samples -- the recursion's 2 m + 4 dependent shuffle chains, not the bytes in flight, bound the half-warp forms at
// full history (profiles/r2_lbfgs_state_select_c5.md).  Here a lane holds 16 coordinates (four float4 chunks): a dot is
// 16 FMAs in four independent chains and TWO shuffle steps, a warp instruction covers eight samples (about a third of the
// instructions per sample), and no history row occupies a register across the recursion: one-warp CTAs of 41 KB, five
// per SM, each issuing its 2 len plane copies at once (lane t copies plane t: parallel issue) and waiting on one mbarrier.
// Physical planes are copied as stored (sample i's logical pair l is plane (head_i + l) mod m, resolved once per lane
// into a row offset); a sample's slots beyond len_i read a row of zeros.  When not all eight samples of the warp are
// active the copies are per sample and row (256 bytes) so that stationary samples cost no traffic.
// Needs d % 4 == 0 and 32 < d <= 64; FULL: d = 64 (no chunk predicates).
constexpr int QS = 8;                                     // samples per warp
struct RowQ { float4 v[4]; };
__device__ __forceinline__ float quad_sum(float v) {      // over the 4 lanes of a sample (all 32 lanes call)
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}
__device__ __forceinline__ float quad_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
  return v;
}
__device__ __forceinline__ float dotq(const RowQ &a, const RowQ &b) {
  float acc[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) acc[k] = fmaf(a.v[k].x, b.v[k].x, fmaf(a.v[k].y, b.v[k].y, fmaf(a.v[k].z, b.v[k].z, a.v[k].w * b.v[k].w)));
  return quad_sum((acc[0] + acc[1]) + (acc[2] + acc[3]));
}
__device__ __forceinline__ float pdotq(const RowQ &a, const RowQ &b) {   // this lane's part of a dot product
  float acc[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) acc[k] = fmaf(a.v[k].x, b.v[k].x, fmaf(a.v[k].y, b.v[k].y, fmaf(a.v[k].z, b.v[k].z, a.v[k].w * b.v[k].w)));
  return (acc[0] + acc[1]) + (acc[2] + acc[3]);
}
__device__ __forceinline__ void quad_sum2(float &u, float &v) {        // two reductions, their shuffles interleaved
  const float u1 = __shfl_xor_sync(0xffffffffu, u, 1), v1 = __shfl_xor_sync(0xffffffffu, v, 1);
  u += u1; v += v1;
  const float u2 = __shfl_xor_sync(0xffffffffu, u, 2), v2 = __shfl_xor_sync(0xffffffffu, v, 2);
  u += u2; v += v2;
}
__device__ __forceinline__ void quad_sum3(float &u, float &v, float &w) {
  const float u1 = __shfl_xor_sync(0xffffffffu, u, 1), v1 = __shfl_xor_sync(0xffffffffu, v, 1), w1 = __shfl_xor_sync(0xffffffffu, w, 1);
  u += u1; v += v1; w += w1;
  const float u2 = __shfl_xor_sync(0xffffffffu, u, 2), v2 = __shfl_xor_sync(0xffffffffu, v, 2), w2 = __shfl_xor_sync(0xffffffffu, w, 2);
  u += u2; v += v2; w += w2;
}
__device__ __forceinline__ void axpyq(RowQ &r, float c, const RowQ &v) {
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    r.v[k].x = fmaf(c, v.v[k].x, r.v[k].x); r.v[k].y = fmaf(c, v.v[k].y, r.v[k].y);
    r.v[k].z = fmaf(c, v.v[k].z, r.v[k].z); r.v[k].w = fmaf(c, v.v[k].w, r.v[k].w);
  }
}
// Register k of lane q holds float4 chunk q + 4 ((k + odd) mod 4) of the row, odd = parity of the sample's slot: the two
// samples a quarter-warp reads with one LDS.128 then hit different banks (their rows are 64 words apart).  As addresses:
// chunks k = 0, 1, 2 sit at c0, c0 + 4, c0 + 8 (c0 = q + 4 odd) and k = 3 at c0 + k3 (k3 = 12 or -4): two adds per row.
struct QuadMap { int c0, k3, d4; };
template <bool FULL>
__device__ __forceinline__ RowQ ld_rowq(const float *row, const QuadMap &mp) {   // global or shared, 16-byte aligned
  const float4 *b = reinterpret_cast<const float4 *>(row) + mp.c0;
  RowQ r;
  if constexpr (FULL) { r.v[0] = b[0]; r.v[1] = b[4]; r.v[2] = b[8]; r.v[3] = b[mp.k3]; }
  else {
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    r.v[0] = (mp.c0 < mp.d4) ? b[0] : z; r.v[1] = (mp.c0 + 4 < mp.d4) ? b[4] : z;
    r.v[2] = (mp.c0 + 8 < mp.d4) ? b[8] : z; r.v[3] = (mp.c0 + mp.k3 < mp.d4) ? b[mp.k3] : z;
  }
  return r;
}
template <bool FULL>
__device__ __forceinline__ void st_rowq(float *row, const QuadMap &mp, const RowQ &r) {
  float4 *b = reinterpret_cast<float4 *>(row) + mp.c0;
  if (FULL || mp.c0 < mp.d4) b[0] = r.v[0];
  if (FULL || mp.c0 + 4 < mp.d4) b[4] = r.v[1];
  if (FULL || mp.c0 + 8 < mp.d4) b[8] = r.v[2];
  if (FULL || mp.c0 + mp.k3 < mp.d4) b[mp.k3] = r.v[3];
}
// history row out of shared memory (byte address in the shared window).  volatile: the three passes of the recursion read
// every row again on purpose -- left to itself the compiler keeps all 2 m rows live from the first pass on and spills them
__device__ __forceinline__ float4 lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
template <bool FULL>
__device__ __forceinline__ RowQ ld_rowq_sh(uint32_t row, const QuadMap &mp) {
  const uint32_t b = row + 16u * mp.c0;
  RowQ r;
  if constexpr (FULL) { r.v[0] = lds128(b); r.v[1] = lds128(b + 64u); r.v[2] = lds128(b + 128u); r.v[3] = lds128(b + 16 * mp.k3); }
  else {
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    r.v[0] = (mp.c0 < mp.d4) ? lds128(b) : z; r.v[1] = (mp.c0 + 4 < mp.d4) ? lds128(b + 64u) : z;
    r.v[2] = (mp.c0 + 8 < mp.d4) ? lds128(b + 128u) : z; r.v[3] = (mp.c0 + mp.k3 < mp.d4) ? lds128(b + 16 * mp.k3) : z;
  }
  return r;
}
__device__ __forceinline__ RowQ zeroq() { RowQ r; r.v[0] = r.v[1] = r.v[2] = r.v[3] = make_float4(0.f, 0.f, 0.f, 0.f); return r; }
__device__ __forceinline__ RowQ subq(const RowQ &a, const RowQ &b) {
  RowQ r;
#pragma unroll
  for (int k = 0; k < 4; ++k) r.v[k] = make_float4(a.v[k].x - b.v[k].x, a.v[k].y - b.v[k].y, a.v[k].z - b.v[k].z, a.v[k].w - b.v[k].w);
  return r;
}

// lbfgs_update_half with four lanes per sample; additionally returns the stored pair and its plane (the recursion that
// follows reads it from shared memory, where these lanes put it)
struct SampleStateQ { RowQ g, x, sv, yv; int len, head, stalled, stored_plane; bool have_x; unsigned bytes; };
template <bool FULL>
__device__ __forceinline__ SampleStateQ lbfgs_update_quad(const State &s, int i, bool in, int q, const QuadMap &mp) {
  const int d = s.d, m = s.m;
  const size_t ro = (size_t)(in ? i : 0) * d;
  SampleStateQ o;
  const int b = in ? s.ls_b[i] : -2;
  o.len = in ? s.hist_len[i] : 0; o.head = in ? s.hist_head[i] : 0; o.stalled = in ? (int)s.stalled[i] : 0;
  o.g = in ? ld_rowq<FULL>(s.g + ro, mp) : zeroq();
  o.x = zeroq(); o.have_x = false; o.bytes = 0u; o.stored_plane = -1;
  const bool acc = b >= 0;
  RowQ x = o.x, xt = o.x, gn = o.x;
  if (acc) { x = ld_rowq<FULL>(s.x + ro, mp); xt = ld_rowq<FULL>(s.xt + ro, mp); gn = ld_rowq<FULL>(s.gn + ro, mp); }
  o.sv = subq(xt, x); o.yv = subq(o.g, gn);
  const float sy = dotq(o.sv, o.yv), ss = dotq(o.sv, o.sv), yy = dotq(o.yv, o.yv);   // executed by all 32 lanes
  if (acc) {
    const float thr = 1e-10f * sqrtf(ss) * sqrtf(yy);
    o.bytes = 5u * d * 4u;
    if (sy > thr) {
      int ph;
      if (o.len == m) { ph = o.head; o.head = (o.head + 1 == m) ? 0 : o.head + 1; }
      else { ph = o.head + o.len; if (ph >= m) ph -= m; o.len += 1; }
      const size_t off = ((size_t)ph * s.hplane + (size_t)i * d);
      st_rowq<FULL>(s.S + off, mp, o.sv);
      st_rowq<FULL>(s.Y + off, mp, o.yv);
      if (q == 0) { s.hist_len[i] = o.len; s.hist_head[i] = o.head; }
      o.bytes += 2u * d * 4u;
      o.stored_plane = ph;
    }
    st_rowq<FULL>(s.x + ro, mp, xt);
    st_rowq<FULL>(s.g + ro, mp, gn);
    if (q == 0) s.f[i] = s.ft[i];
    o.g = gn; o.x = xt; o.have_x = true;
  } else if (b == -1) {
    if (o.len == 0) { o.stalled = 1; if (q == 0) s.stalled[i] = 1; }
    else { o.len = 0; o.head = 0; if (q == 0) { s.hist_len[i] = 0; s.hist_head[i] = 0; } }
  }
  return o;
}

// shared memory: [m planes of S][64 zeros][m planes of Y][64 zeros][mbarrier]; a plane = QS rows of d floats
__host__ __device__ inline size_t quad_smem_bytes(int m, int d) { return (size_t)2 * ((size_t)m * QS * d + 64) * 4 + 16; }

template <int MM, int MODE, bool FULL>
__global__ void __launch_bounds__(32, 5) k_lbfgs_step_quad(State s, Hyper h) {
  extern __shared__ __align__(128) unsigned char quad_smem[];
  const int lane = threadIdx.x, sidx = lane >> 2, q = lane & 3;
  const int d = FULL ? 64 : s.d, m = s.m, N = s.N;
  const int i0 = blockIdx.x * QS, i = i0 + sidx;
  const int plane_floats = QS * d;
  const int yoff = m * plane_floats + 64;                 // Y array relative to S array (floats)
  const int zoff = m * plane_floats;                      // the row of zeros of either array, relative to its start
  float *hS = reinterpret_cast<float *>(quad_smem);
  float *hY = hS + yoff;
  uint64_t *bar = reinterpret_cast<uint64_t *>(hY + yoff);
  QuadMap mp;
  mp.c0 = q + 4 * (sidx & 1); mp.k3 = (sidx & 1) ? -4 : 12; mp.d4 = d >> 2;
  if (lane == 0) { mbar_init(bar, 1); mbar_fence_init(); }
  hS[zoff + lane] = 0.f; hS[zoff + lane + 32] = 0.f; hY[zoff + lane] = 0.f; hY[zoff + lane + 32] = 0.f;
  if (blockIdx.x == 0 && lane == 0) {
    s.ctrl->ls_cnt[1] = 0; s.ctrl->ls_cnt[2] = 0; s.ctrl->fd_cnt = 0;
    if (MODE != STEP_ALONE) s.ctrl->fmax_enc = 0u;
  }
  __syncwarp();
  const bool in = i < N;
  const size_t ro = (size_t)(in ? i : 0) * d;
  RowQ g, x = zeroq(), sv = zeroq(), yv = zeroq();
  int stalled_i, len_i, head_i, stored_plane = -1;
  bool have_x = false;
  unsigned upd_bytes = 0u;
  if constexpr (MODE == STEP_UPDATE) {
    const SampleStateQ u = lbfgs_update_quad<FULL>(s, i, in, q, mp);
    g = u.g; x = u.x; have_x = u.have_x; stalled_i = u.stalled; len_i = u.len; head_i = u.head; upd_bytes = u.bytes;
    sv = u.sv; yv = u.yv; stored_plane = u.stored_plane;
  } else {
    g = in ? ld_rowq<FULL>(s.g + ro, mp) : zeroq();
    stalled_i = s.stalled[in ? i : 0]; len_i = s.hist_len[in ? i : 0]; head_i = s.hist_head[in ? i : 0];
  }
  float ga = 0.f;
#pragma unroll
  for (int k = 0; k < 4; ++k) ga = fmaxf(ga, fmaxf(fmaxf(fabsf(g.v[k].x), fabsf(g.v[k].y)), fmaxf(fabsf(g.v[k].z), fabsf(g.v[k].w))));
  const float ginf = quad_max(ga);
  // (i) stationary (Eq. 3's gradient test) or stalled: no work, no evaluations (R-6)
  const bool act = in && !(stalled_i || !(ginf >= h.eps_grad));
  int len = act ? len_i : 0;
  const int len_read = len;
  const int head = act ? head_i : 0;
  // ---- history into shared memory ------------------------------------------------------------------------------------
  // planes a sample reads: 0 .. len - 1 while its ring has not wrapped (head = 0), all m afterwards
  const int need = (len == 0) ? 0 : (head == 0 ? len : m);
  int L = need;                                            // planes to copy: max over the warp
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) L = max(L, __shfl_xor_sync(0xffffffffu, L, o));
  const unsigned actmask = __ballot_sync(0xffffffffu, act);
  const int nvalid = min(QS, N - i0);
  const bool dense = actmask == (nvalid == QS ? 0xffffffffu : ((1u << (4 * nvalid)) - 1u));
  if (L > 0) {
    if (dense) {                                           // every sample of the warp is active: one copy per plane and array
      const uint32_t pbytes = (uint32_t)nvalid * d * 4u;
      if (lane == 0) mbar_expect_tx(bar, 2u * L * pbytes);
      __syncwarp();
      if (lane < 2 * L) {
        const int ph = lane >> 1;
        const float *src = ((lane & 1) ? s.Y : s.S) + (size_t)ph * s.hplane + (size_t)i0 * d;
        bulk_g2s(((lane & 1) ? hY : hS) + (size_t)ph * plane_floats, src, pbytes, bar);
      }
    } else {                                               // per active sample and plane (lane q of the sample takes planes q, q + 4, ..)
      unsigned tot = (q == 0) ? (unsigned)need * 2u * d * 4u : 0u;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      if (lane == 0) mbar_expect_tx(bar, tot);
      __syncwarp();
      for (int ph = q; ph < need; ph += 4) {
        const size_t off = (size_t)ph * s.hplane + (size_t)i * d;
        bulk_g2s(hS + (size_t)ph * plane_floats + sidx * d, s.S + off, (uint32_t)d * 4u, bar);
        bulk_g2s(hY + (size_t)ph * plane_floats + sidx * d, s.Y + off, (uint32_t)d * 4u, bar);
      }
    }
  }
  if (act && !have_x) x = ld_rowq<FULL>(s.x + ro, mp);
  // warp-aggregated append of the searching samples to line-search worklist 0, and the byte counter
  const unsigned heads = actmask & 0x11111111u;
  const int my_slot = __popc(heads & ((1u << lane) - 1u));
  unsigned bytes = (in && q == 0) ? upd_bytes + (2u * d + (act ? 2u * (unsigned)len_read * d + 2u * d : 0u)) * 4u : 0u;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
  int base = 0;
  if (lane == 0) {
    if (heads) base = atomicAdd(&s.ctrl->ls_cnt[0], __popc(heads));
    if (bytes) atomicAdd(&s.ctrl->evals[7], (unsigned long long)bytes);
  }
  RowQ gam;
#pragma unroll
  for (int k = 0; k < 4; ++k) gam.v[k] = make_float4(-g.v[k].x, -g.v[k].y, -g.v[k].z, -g.v[k].w);
  RowQ p = zeroq(), xt = zeroq();
  bool restart = false;
  float t0 = 0.f, dec = 0.f;
  const uint32_t aS = smem_u32(hS), aY = smem_u32(hY);
  // row offset (bytes, relative to the array) of logical pair l of this sample: plane (head + l) mod m of its slot, or
  // the row of zeros beyond len
  int roff[MM];
#pragma unroll
  for (int l = 0; l < MM; ++l) {
    int ph = head + l; if (ph >= m) ph -= m;
    roff[l] = 4 * ((l < len_read) ? ph * plane_floats + sidx * d : zoff);
  }
  if (L > 0) mbar_wait(bar, 0);
  if constexpr (MODE == STEP_UPDATE) {
    // the pair this launch has just stored: its rows go to shared memory from the registers that hold them (the copy of
    // that plane may have read the row before or after the global store).  A lane reads back only chunks it wrote.
    if (act && stored_plane >= 0) {
      st_rowq<FULL>(hS + (size_t)stored_plane * plane_floats + sidx * d, mp, sv);
      st_rowq<FULL>(hY + (size_t)stored_plane * plane_floats + sidx * d, mp, yv);
    }
  }
  if (actmask) {
    const float gn2 = dotq(g, g);
    // Straight-line code over all MM slots (this form runs when the rings are full or nearly so): slots beyond len read
    // the row of zeros with rho = 0 and contribute nothing, and no shuffle sits under a branch.
    // The recursion advances TWO pairs per dependent step.  First loop, pairs (l, l - 1), l odd, newest first:
    //   alpha_l = rho_l s_l.q,   alpha_{l-1} = rho_{l-1} s_{l-1}.(q - alpha_l y_l) = rho_{l-1} (s_{l-1}.q - alpha_l b_l),
    // b_l = s_{l-1}.y_l -- both dots are taken with the same q, so their shuffle reductions overlap; second loop, pairs
    // (l - 1, l): beta_{l-1} = rho_{l-1} y_{l-1}.r, beta_l = rho_l (y_l.r + (alpha_{l-1} - beta_{l-1}) b_l).  The b_l do not
    // depend on q or r and are computed with the rho_l up front, where every dot is independent of the others.
    static_assert(MM % 2 == 0, "pairs");
    float rho[MM], al[MM], bq[MM / 2];
#pragma unroll
    for (int l = 1; l < MM; l += 2) {
      const RowQ S0 = ld_rowq_sh<FULL>(aS + roff[l - 1], mp), Y0 = ld_rowq_sh<FULL>(aY + roff[l - 1], mp);
      const RowQ S1 = ld_rowq_sh<FULL>(aS + roff[l], mp), Y1 = ld_rowq_sh<FULL>(aY + roff[l], mp);
      float sy0 = pdotq(S0, Y0), sy1 = pdotq(S1, Y1), b = pdotq(S0, Y1);
      quad_sum3(sy0, sy1, b);
      rho[l - 1] = (l - 1 < len_read) ? 1.0f / sy0 : 0.0f;
      rho[l] = (l < len_read) ? 1.0f / sy1 : 0.0f;
      bq[l >> 1] = b;
    }
    RowQ r = gam;
#pragma unroll
    for (int l = MM - 1; l >= 1; l -= 2) {
      const RowQ S1 = ld_rowq_sh<FULL>(aS + roff[l], mp), S0 = ld_rowq_sh<FULL>(aS + roff[l - 1], mp);
      float a1 = pdotq(S1, r), a0 = pdotq(S0, r);
      quad_sum2(a1, a0);
      al[l] = rho[l] * a1;
      al[l - 1] = rho[l - 1] * fmaf(-al[l], bq[l >> 1], a0);
      axpyq(r, -al[l], ld_rowq_sh<FULL>(aY + roff[l], mp));
      axpyq(r, -al[l - 1], ld_rowq_sh<FULL>(aY + roff[l - 1], mp));
    }
    {
      // H0 = (s.y / y.y) I of the newest pair: its row offset is arithmetic (a select over rho[] and roff[] by len would
      // put both arrays in local memory), and s.y is taken again rather than looked up
      int phn = head + len_read - 1; if (phn >= m) phn -= m;
      const int roff_n = 4 * ((len_read > 0) ? phn * plane_floats + sidx * d : zoff);
      const RowQ Yn = ld_rowq_sh<FULL>(aY + roff_n, mp), Sn = ld_rowq_sh<FULL>(aS + roff_n, mp);
      float yy = pdotq(Yn, Yn), syn = pdotq(Sn, Yn);
      quad_sum2(yy, syn);
      if (len_read > 0) {
        const float h0 = syn / yy;
#pragma unroll
        for (int k = 0; k < 4; ++k) { r.v[k].x *= h0; r.v[k].y *= h0; r.v[k].z *= h0; r.v[k].w *= h0; }
      }
    }
#pragma unroll
    for (int l = 1; l < MM; l += 2) {
      const RowQ Y0 = ld_rowq_sh<FULL>(aY + roff[l - 1], mp), Y1 = ld_rowq_sh<FULL>(aY + roff[l], mp);
      float c0 = pdotq(Y0, r), c1 = pdotq(Y1, r);
      quad_sum2(c0, c1);
      const float d0 = al[l - 1] - rho[l - 1] * c0;
      const float d1 = al[l] - rho[l] * fmaf(d0, bq[l >> 1], c1);
      axpyq(r, d0, ld_rowq_sh<FULL>(aS + roff[l - 1], mp));
      axpyq(r, d1, ld_rowq_sh<FULL>(aS + roff[l], mp));
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) p.v[k] = make_float4(-r.v[k].x, -r.v[k].y, -r.v[k].z, -r.v[k].w);
    const float gp = dotq(gam, p);
    if (len > 0 && !(gp < 0.0f)) { restart = true; len = 0; }   // not a descent direction for phi = -f: steepest restart
    if (len_read == 0 || restart) p = g;                         // p = -gam
    // (iii) first trial step; (iv) trial point projected on Theta, Armijo linear term gamma.(x_t - x)
    t0 = (len > 0) ? 1.0f : fminf(1.0f, 1.0f / sqrtf(gn2));
    const RowQ lo = ld_rowq<FULL>(s.lo, mp), hi = ld_rowq<FULL>(s.hi, mp);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      xt.v[k].x = clipf(fmaf(t0, p.v[k].x, x.v[k].x), lo.v[k].x, hi.v[k].x);
      xt.v[k].y = clipf(fmaf(t0, p.v[k].y, x.v[k].y), lo.v[k].y, hi.v[k].y);
      xt.v[k].z = clipf(fmaf(t0, p.v[k].z, x.v[k].z), lo.v[k].z, hi.v[k].z);
      xt.v[k].w = clipf(fmaf(t0, p.v[k].w, x.v[k].w), lo.v[k].w, hi.v[k].w);
    }
    dec = dotq(gam, subq(xt, x));
  }
  if (in) {
    if (act) {
      st_rowq<FULL>(s.xt + ro, mp, xt);
      st_rowq<FULL>(s.p + ro, mp, p);
      if (q == 0) {
        s.dec[i] = dec; s.tcur[i] = t0; s.ls_b[i] = -1;
        if (restart) { s.hist_len[i] = 0; s.hist_head[i] = 0; }
      }
    } else {
      st_rowq<FULL>(s.p + ro, mp, zeroq());
      if (q == 0) s.ls_b[i] = -2;
    }
  }
  base = __shfl_sync(0xffffffffu, base, 0);
  if (act && q == 0) s.ls_list[0][base + my_slot] = i;
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
static cudaError_t launch_step_one(const State &s, const Hyper &h, int grid, int hrows, cudaStream_t st) {
  hrows = SH ? std::max(1, std::min(hrows, MM)) : MM;
  const size_t sh = SH ? (size_t)DIR_WARPS * 2 * 2 * hrows * 16 * sizeof(float4) : 0;
  if (SH) {
    static bool configured = false;
    if (!configured) {
      const size_t shmax = (size_t)DIR_WARPS * 2 * 2 * MM * 16 * sizeof(float4);
      cudaError_t e = cudaFuncSetAttribute(k_lbfgs_step<MM, VEC, MODE, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmax);
      if (e != cudaSuccess) return e;
      e = cudaFuncSetAttribute(k_lbfgs_step<MM, VEC, MODE, SH>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
      if (e != cudaSuccess) return e;
      configured = true;
    }
  }
  k_lbfgs_step<MM, VEC, MODE, SH><<<grid, DIR_WARPS * 32, sh, st>>>(s, h, hrows);
  return cudaGetLastError();
}
template <int MM, bool VEC, bool SH>
static cudaError_t launch_step_mode(const State &s, const Hyper &h, int mode, int grid, int hrows, cudaStream_t st) {
  if (mode == STEP_FIRST) return launch_step_one<MM, VEC, STEP_FIRST, false>(s, h, grid, hrows, st);   // (empty history: nothing to stage)
  if (mode == STEP_UPDATE) return launch_step_one<MM, VEC, STEP_UPDATE, SH>(s, h, grid, hrows, st);
  return launch_step_one<MM, VEC, STEP_ALONE, SH>(s, h, grid, hrows, st);
}
template <int MM>
static cudaError_t launch_step_mm(const State &s, const Hyper &h, int mode, bool staged, int grid, int hrows, cudaStream_t st) {
  const bool vec = (s.d & 3) == 0;
  if (!vec) return launch_step_mode<MM, false, false>(s, h, mode, grid, hrows, st);
  if (!staged) return launch_step_mode<MM, true, false>(s, h, mode, grid, hrows, st);
  return launch_step_mode<MM, true, true>(s, h, mode, grid, hrows, st);
}
static int g_step_quad = 1;        // CHISAO_STEP_QUAD in the environment: 0 never, 1 where the register form would run (default), 2 also for it <= m
template <int MM, int MODE, bool FULL>
static cudaError_t launch_quad_one(const State &s, const Hyper &h, cudaStream_t st) {
  const size_t sh = quad_smem_bytes(s.m, s.d);
  static size_t configured = 0;
  if (sh > configured) {
    cudaError_t e = cudaFuncSetAttribute(k_lbfgs_step_quad<MM, MODE, FULL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_lbfgs_step_quad<MM, MODE, FULL>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    configured = sh;
  }
  k_lbfgs_step_quad<MM, MODE, FULL><<<(s.N + QS - 1) / QS, 32, sh, st>>>(s, h);
  return cudaGetLastError();
}
template <int MM>
static cudaError_t launch_quad_mm(const State &s, const Hyper &h, int mode, cudaStream_t st) {
  if (s.d == 64) return mode == STEP_UPDATE ? launch_quad_one<MM, STEP_UPDATE, true>(s, h, st) : launch_quad_one<MM, STEP_ALONE, true>(s, h, st);
  return mode == STEP_UPDATE ? launch_quad_one<MM, STEP_UPDATE, false>(s, h, st) : launch_quad_one<MM, STEP_ALONE, false>(s, h, st);
}
// `it`: iteration of the cycle (0 for the stand-alone unit): after it - 1 updates a history holds at most it - 1 pairs
cudaError_t launch_lbfgs_step(const State &s, const Hyper &h, int mode, int it, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  static bool env_read = false;
  if (!env_read) {
    g_step_regs = getenv("CHISAO_STEP_REGS") != nullptr;
    if (const char *e = getenv("CHISAO_STEP_QUAD")) g_step_quad = atoi(e);
    env_read = true;
  }
  const int per_block = DIR_WARPS * 2, grid = (s.N + per_block - 1) / per_block;
  const bool staged = !g_step_regs && mode == STEP_UPDATE && it - 1 < s.m;   // the ring cannot be full yet
  // four lanes per sample, history planes bulk-copied to shared memory: the form for full histories at 32 < d <= 64
  if (mode != STEP_FIRST && (s.d & 3) == 0 && s.d > 32 && (g_step_quad == 2 || (g_step_quad == 1 && !staged))) {
    if (s.m <= 4) return launch_quad_mm<4>(s, h, mode, st);
    if (s.m <= 8) return launch_quad_mm<8>(s, h, mode, st);
    if (s.m <= 10) return launch_quad_mm<10>(s, h, mode, st);
    return launch_quad_mm<16>(s, h, mode, st);
  }
  const int hrows = staged ? it - 1 : s.m;                  // pairs a history can hold in this launch
  if (s.m <= 4) return launch_step_mm<4>(s, h, mode, staged, grid, hrows, st);
  if (s.m <= 8) return launch_step_mm<8>(s, h, mode, staged, grid, hrows, st);
  if (s.m <= 10) return launch_step_mm<10>(s, h, mode, staged, grid, hrows, st);
  return launch_step_mm<16>(s, h, mode, staged, grid, hrows, st);
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
