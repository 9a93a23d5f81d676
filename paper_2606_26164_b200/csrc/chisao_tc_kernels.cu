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

// ---- FD stencil on the QUAD fp16 form: the operand image of a tile is built ONCE per warp ------------------------------------
// At 32 < d <= 64 the 128 points of a group are the 2d stencil points of ONE sample: every thread's operand row is the
// sample's 2^k (x - c) with one coordinate moved by +-h.  Instead of 128 threads each subtracting, scaling and splitting
// the same 64 numbers (quad_write_a16: ~450 instructions per thread and tile, which bound the kernel), lane l of every warp
// does coordinates l and l + 32, the warp's 64 hi and 64 lo halves meet in 256 bytes of shared memory, every lane reads
// the packed row back (16 broadcast LDS.128), patches the word that holds its own coordinate and stores the row to its TMEM
// lane.  The scale 2^k is taken from max_c |x_c - c_c| + h, a bound on every point of the stencil.  Same pipeline as
// tc_quad_run16<DEEP>: rows are requested three tiles ahead, the image of tile n + 2 is built while the MMAs of tile
// n + 1 run.
struct Fd16Pre { float xa, xb; int i; bool valid; };
template <class Finish>
__device__ __forceinline__ void tc_quad_fd16(const TcObj &o, const TcSmem &sm, int t, int ntiles, const FdArgs &a, int cnt, Finish finish) {
  const int warp = __shfl_sync(0xffffffffu, t >> 5, 0);   // provably warp-uniform role index
  if (warp == TC_PTS / 32) {
    if (t == TC_PTS) {
      mbar_expect_tx(sm.bbar(0), TC_REC_BYTES);
      bulk_g2s(sm.B(0), o.recs, TC_REC_BYTES, sm.bbar(0));
    }
    return;
  }
  if (warp > TC_PTS / 32) { quad_issuer16(sm, tcx_tiles_of_cta(ntiles)); return; }
  const uint32_t tm = *sm.tmem();
  const int g = t >> 7, lane = t & 31, w4 = (t >> 5) & 3, tl = t & 127, d = a.d;
  const int slot = tl, j = slot >> 1;
  const bool lane_pt = tl < 2 * d;                          // the thread has a stencil point (d < 64: the last lanes idle)
  const uint32_t lane_base = tm + ((uint32_t)(w4 * 32) << 16) + (uint32_t)(g * 256);
  const int ntc = tcx_tiles_of_cta(ntiles), stride = (int)gridDim.x;
  mbar_wait(sm.bbar(0), 0);                                 // W images and c have landed
  const float *mu = sm.B(0) + 2 * TC_D * TC_D;              // (zero beyond d)
  const float mua = mu[lane], mub = mu[lane + 32], muj = mu[j];
  uint16_t *stage = reinterpret_cast<uint16_t *>(sm.scratch()) + (t >> 5) * 128;   // the warp's 64 hi + 64 lo halves
  // The worklist entry of a tile is requested one tile before its row (a dependent index -> row chain issued in one go
  // stalls the warp at the address computation for a whole L2 round trip: in-order issue), the row two tiles before the
  // operand build that consumes it.
  auto pre_idx = [&](int tile) -> int {
    const int e = tile * 2 + g;
    return (tile < ntiles && e < cnt) ? (a.list ? a.list[e] : e) : -1;
  };
  auto pre_row = [&](int idx) -> Fd16Pre {                  // the sample of this group: two coordinates per lane
    Fd16Pre p;
    p.valid = idx >= 0;
    p.i = p.valid ? idx : 0;
    const float *row = a.X + (size_t)p.i * d;
    p.xa = (p.valid && lane < d) ? row[lane] : 0.f;
    p.xb = (p.valid && lane + 32 < d) ? row[lane + 32] : 0.f;
    return p;
  };
  auto halves = [](float v, uint32_t &hi, uint32_t &lo) {
    const __half hh = __float2half_rn(v);
    hi = (uint32_t)__half_as_ushort(hh);
    lo = (uint32_t)__half_as_ushort(__float2half_rn(v - __half2float(hh)));
  };
  auto build = [&](const Fd16Pre &p, int buf, FdCtx &c) -> float {
    const float va = p.xa - mua, vb = p.xb - mub;
    const float vmax = warp_max(fmaxf(fabsf(va), fabsf(vb))) + a.h;
    int k = 3 - ((int)((__float_as_uint(vmax) >> 23) & 0xffu) - 127);
    k = min(max(k, -30), 40);
    const float sc = __uint_as_float((uint32_t)(k + 127) << 23);
    uint32_t ha, la, hb, lb;
    halves(va * sc, ha, la); halves(vb * sc, hb, lb);
    __syncwarp();                                           // the previous image has been read back by every lane
    stage[lane] = (uint16_t)ha; stage[lane + 32] = (uint16_t)hb; stage[64 + lane] = (uint16_t)la; stage[96 + lane] = (uint16_t)lb;
    __syncwarp();
    uint32_t h[32], l[32];
    const uint4 *sv = reinterpret_cast<const uint4 *>(stage);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const uint4 u = sv[q], v = sv[8 + q];
      h[4 * q] = u.x; h[4 * q + 1] = u.y; h[4 * q + 2] = u.z; h[4 * q + 3] = u.w;
      l[4 * q] = v.x; l[4 * q + 1] = v.y; l[4 * q + 2] = v.z; l[4 * q + 3] = v.w;
    }
    // the thread's own coordinate j = 16 w4 + lane / 2 sits in lane j mod 32 (first or second coordinate of that lane)
    const float xj = __shfl_sync(0xffffffffu, (w4 < 2) ? p.xa : p.xb, j & 31);
    c.i = p.i; c.valid = p.valid && lane_pt;
    c.xj = c.valid ? xj : 0.f;
    c.xp = c.valid ? ((slot & 1) ? xj - a.h : xj + a.h) : 0.f;
    uint32_t hj, lj;
    halves((c.xp - muj) * sc, hj, lj);
    // its halves go into word j / 2 = 8 w4 + lane / 4 of the hi and of the lo image, half j & 1 (static register indices:
    // one warp-uniform branch per warp of the group, eight candidate words each)
    if (c.valid) {
      const int tw = lane >> 2;
      const uint32_t keep = (j & 1) ? 0x0000FFFFu : 0xFFFF0000u, sh = (j & 1) ? 16u : 0u;
#pragma unroll
      for (int wq = 0; wq < 4; ++wq)
        if (w4 == wq) {
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const bool me = tw == q;
            h[8 * wq + q] = me ? ((h[8 * wq + q] & keep) | (hj << sh)) : h[8 * wq + q];
            l[8 * wq + q] = me ? ((l[8 * wq + q] & keep) | (lj << sh)) : l[8 * wq + q];
          }
        }
    }
    const uint32_t acol = lane_base + (uint32_t)(64 * buf);
    {
      uint32_t v16[16];
#pragma unroll
      for (int q = 0; q < 16; ++q) v16[q] = h[q];
      tc_st16u(acol, v16);
#pragma unroll
      for (int q = 0; q < 16; ++q) v16[q] = h[16 + q];
      tc_st16u(acol + 16, v16);
#pragma unroll
      for (int q = 0; q < 16; ++q) v16[q] = l[q];
      tc_st16u(acol + 32, v16);
#pragma unroll
      for (int q = 0; q < 16; ++q) v16[q] = l[16 + q];
      tc_st16u(acol + 48, v16);
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncwarp();
    if (lane == 0) mbar_arrive(buf ? sm.dbar(g) : sm.xbar(g));
    return __uint_as_float((uint32_t)(127 - 2 * (k + o.quad_ws)) << 23);
  };
  FdCtx c0{}, c1{}, c2{};
  const int b0 = (int)blockIdx.x;
  Fd16Pre P = pre_row(pre_idx(b0));
  float u0 = build(P, 0, c0), u1 = 0.f, u2 = 0.f;
  if (ntc > 1) { P = pre_row(pre_idx(b0 + stride)); u1 = build(P, 1, c1); }
  Fd16Pre Pa = pre_row(pre_idx(b0 + 2 * stride)), Pb = pre_row(pre_idx(b0 + 3 * stride));   // rows of tiles it + 2, it + 3
  int idx_n = pre_idx(b0 + 4 * stride);                                                       // entry of tile it + 4
  // one tile; Px holds the row of tile it + 2 on entry and the (requested) row of tile it + 4 on exit.  The loop below
  // alternates between two such registers sets instead of rotating them: a register move of a value whose load is
  // still in flight waits for the load (21 % of the kernel's stall samples sat on that move).
  auto step = [&](int it, Fd16Pre &Px) {
    const int tile = (int)blockIdx.x + it * stride, st = it & 1;
    mbar_wait(sm.cbar(2 * g + st), (it >> 1) & 1);          // MMAs of tile `it` retired: image st and accumulator stage st are ours
    asm volatile("tcgen05.fence::after_thread_sync;");
    float q0 = 0.f, q1 = 0.f, q2 = 0.f, q3 = 0.f;
    {
      uint32_t r[64];
      const uint32_t ta = lane_base + 128 + (uint32_t)(64 * st);
      tc_ld16s64(ta, r, 0); tc_ld16s64(ta + 16, r, 1); tc_ld16s64(ta + 32, r, 2); tc_ld16s64(ta + 48, r, 3);
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      asm volatile("tcgen05.fence::before_thread_sync;");
      __syncwarp();
      if (lane == 0) mbar_arrive(sm.rdbar(2 * g + st));
#pragma unroll
      for (int n = 0; n < 64; n += 4) {
        const float z0 = __uint_as_float(r[n]), z1 = __uint_as_float(r[n + 1]), z2 = __uint_as_float(r[n + 2]),
                    z3 = __uint_as_float(r[n + 3]);
        q0 = fmaf(z0, z0, q0); q1 = fmaf(z1, z1, q1); q2 = fmaf(z2, z2, q2); q3 = fmaf(z3, z3, q3);
      }
    }
    if (it + 2 < ntc) u2 = build(Px, st, c2);
    finish(tile, -0.5f * u0 * ((q0 + q1) + (q2 + q3)), c0);
    c0 = c1; u0 = u1; c1 = c2; u1 = u2;
    Px = pre_row(idx_n);                                     // tile it + 4: consumed two iterations from now, from this same set
    idx_n = pre_idx(tile + 5 * stride);
  };
  for (int it = 0; it < ntc; it += 2) {
    step(it, Pa);
    if (it + 1 < ntc) step(it + 1, Pb);
  }
}

template <class Finish>
__device__ __forceinline__ void tc_rff_fd32(const TcObj &o, const TcSmem &sm, int t, int ntiles, const FdArgs &a, int cnt, Finish finish) {
  const int ntc = tcx_tiles_of_cta(ntiles);
  const int warp = __shfl_sync(0xffffffffu, t >> 5, 0);   // provably warp-uniform role index
  if (warp == TC_PTS / 32) {
    if (t == TC_PTS) {
      mbar_expect_tx(sm.bbar(0), RFF_REC_BYTES);
      bulk_g2s(sm.Bx(0, 0), o.recs, RFF_REC_BYTES, sm.bbar(0));
    }
    return;
  }
  if (warp > TC_PTS / 32) { rff_issuer(o, sm, ntc); return; }
  mbar_wait(sm.bbar(0), 0);
  const int g = t >> 7, tl = t & 127, lane = t & 31, w4 = (t >> 5) & 3;
  const int slot = tl & 63, j = slot >> 1;                  // j = 16 (w4 & 1) + lane / 2
  unsigned char *wbase = reinterpret_cast<unsigned char *>(sm.Bx(0, 0));
  unsigned char *ximg = wbase + RFF_REC_BYTES + g * RFF_X_BYTES;
  uint16_t *stage = reinterpret_cast<uint16_t *>(sm.scratch()) + (t >> 5) * 128;   // the warp's 4 x 32 halves
  const float S0 = o.rff_S0, U0 = 1.0f / S0;
  const int stride = (int)gridDim.x;
  auto halves4 = [&](float v, uint32_t (&hv)[4]) {
    float n0, n1, n2;
    rff_split(v, S0, U0, n0, n1, n2);
    hv[0] = (uint32_t)__half_as_ushort(__float2half_rn(n0));
    hv[1] = (uint32_t)__half_as_ushort(__float2half_rn(n1));
    hv[2] = (uint32_t)__half_as_ushort(__float2half_rn(n1 * (1.0f / 1024.0f)));
    hv[3] = (uint32_t)__half_as_ushort(__float2half_rn(n2 * (1.0f / 1024.0f)));
  };
  struct Pre { float xc; int i; bool valid; };
  // (the worklist entry is requested one tile before the row: a dependent index -> row chain issued in one go stalls
  // the warp at the address computation, in-order issue)
  auto pre_idx = [&](int tile) -> int {
    const int e = tile * 4 + 2 * g + (w4 >> 1);
    return (tile < ntiles && e < cnt) ? (a.list ? a.list[e] : e) : -1;
  };
  auto pre_row = [&](int idx) -> Pre {                      // coordinate `lane` of the warp's sample
    Pre p;
    p.valid = idx >= 0;
    p.i = p.valid ? idx : 0;
    p.xc = p.valid ? a.X[(size_t)p.i * 32 + lane] : 0.f;
    return p;
  };
  Pre P = pre_row(pre_idx((int)blockIdx.x));
  int idx_n = pre_idx((int)blockIdx.x + stride);
  for (int it = 0; it < ntc; ++it) {
    const int tile = (int)blockIdx.x + it * stride;
    const Pre cur = P;
    uint32_t hv[4];
    halves4(cur.xc, hv);
    __syncwarp();                                           // the previous tile's staged row has been read by every lane
    stage[lane] = (uint16_t)hv[0]; stage[32 + lane] = (uint16_t)hv[1]; stage[64 + lane] = (uint16_t)hv[2]; stage[96 + lane] = (uint16_t)hv[3];
    __syncwarp();
    uint32_t img[4][16];                                    // [image][4 chunks x 4 words]: halves of coordinates 8 kc + 2 w, + 1
    const uint4 *sv = reinterpret_cast<const uint4 *>(stage);
#pragma unroll
    for (int pi = 0; pi < 4; ++pi)
#pragma unroll
      for (int kc = 0; kc < 4; ++kc) {
        const uint4 u = sv[4 * pi + kc];
        img[pi][4 * kc] = u.x; img[pi][4 * kc + 1] = u.y; img[pi][4 * kc + 2] = u.z; img[pi][4 * kc + 3] = u.w;
      }
    const float ssq = warp_sum(cur.xc * cur.xc);
    const float xj = __shfl_sync(0xffffffffu, cur.xc, j);
    FdCtx c;
    c.i = cur.i; c.valid = cur.valid;
    c.xj = c.valid ? xj : 0.f;
    c.xp = c.valid ? ((slot & 1) ? xj - a.h : xj + a.h) : 0.f;
    uint32_t pv[4];
    halves4(c.xp, pv);
#pragma unroll
    for (int kc = 0; kc < 4; ++kc) {
      unsigned char *dst = ximg + kc * 2048 + tl * 16;
#pragma unroll
      for (int pi = 0; pi < 4; ++pi)
        *reinterpret_cast<uint4 *>(dst + 8192 * pi) = make_uint4(img[pi][4 * kc], img[pi][4 * kc + 1], img[pi][4 * kc + 2], img[pi][4 * kc + 3]);
    }
    // own coordinate j: its four halves are stored over the row just written (same thread: program order), chunk j / 8,
    // position j % 8 -- no register of the row is indexed dynamically
    {
      unsigned char *own = ximg + (j >> 3) * 2048 + tl * 16 + (j & 7) * 2;
#pragma unroll
      for (int pi = 0; pi < 4; ++pi) *reinterpret_cast<uint16_t *>(own + 8192 * pi) = (uint16_t)pv[pi];
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.xbar(g));
    const float nrm = c.valid ? (ssq - xj * xj) + c.xp * c.xp : 0.f;
    P = pre_row(idx_n);                                     // tile it + 1: in flight during the chunk loop
    idx_n = pre_idx(tile + 2 * stride);
    const float f = fmaf(-o.rff_s0, nrm, rff_chunks(o, sm, t, it));
    finish(tile, f, c);
  }
}

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
      if constexpr (OBJ == CHISAO_OBJ_GMM_FULL) c.xp = (slot & 1) ? c.xj - a.h : c.xj + a.h;
      // QUAD / RFF: nothing here may touch the loaded values -- the row is requested a tile ahead and patched (below)
      // where the evaluator first consumes it; arithmetic on it here would wait for the loads on the spot
      if constexpr (OBJ != CHISAO_OBJ_GMM_FULL) {
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
  // replace coordinate j by compare-and-select over the whole row: every lane runs the same straight-line code (a
  // dynamically indexed register array would be lowered to a branch tree over j, and the warp-collective tcgen05
  // instructions of the evaluator need every lane on the same path)
  auto patch = [&](FdCtx &c, float (&x)[TC_D]) {
    if constexpr (OBJ != CHISAO_OBJ_GMM_FULL) {
      c.xp = (slot & 1) ? c.xj - a.h : c.xj + a.h;
      if (c.valid) {
#pragma unroll
        for (int q = 0; q < TC_D; ++q) x[q] = (q == j) ? c.xp : x[q];
      } else c.xp = 0.f;
    }
  };
  if constexpr (OBJ == CHISAO_OBJ_QUAD) {
    if (o.f16 && spg == 1) {                               // (d > 32: a group's 128 points are one sample's stencil)
      tc_quad_fd16(o, sm, t, ntiles, a, cnt, finish);
      tc_teardown(sm, t);
      return;
    }
  }
  if constexpr (OBJ == CHISAO_OBJ_RFF) {
    if (d == 32) {                                         // (a warp's 32 points are stencil points of one sample)
      tc_rff_fd32(o, sm, t, ntiles, a, cnt, finish);
      tc_teardown(sm, t);
      return;
    }
  }
  tc_run<OBJ, true>(o, sm, t, ntiles, load, finish, patch);
  tc_teardown(sm, t);
}

struct PtCtx { int i; bool valid; };
template <int OBJ>
__global__ void __launch_bounds__(TC_THREADS, 1) k_eval_points_tc(const TcObj o, const PtArgs a) {
  extern __shared__ __align__(1024) unsigned char tc_smem_raw[];
  const TcSmem sm = tc_carve(tc_smem_raw);
  const int t = threadIdx.x, d = a.d;
  const int cnt = a.count ? *a.count : a.max_count;
  const int ppc = (OBJ != CHISAO_OBJ_GMM_FULL && a.mode == PT_LS_ALL) ? a.tc_pts : TC_PTS;   // worklist entries per CTA
  const int ntiles = (cnt + ppc - 1) / ppc;
  if (blockIdx.x == 0 && t == 0 && a.zero_cnt) *a.zero_cnt = 0;
  if ((int)blockIdx.x >= ntiles) return;
  tc_begin<OBJ>(sm, t);
  if constexpr (OBJ != CHISAO_OBJ_GMM_FULL) {
    if (a.mode == PT_LS_ALL) {
      // every trial b = 0 .. ls_max of the CTA's 256 (or 128) worklist entries in one launch (tc_rounds): round r = trial b
      const int e = (int)blockIdx.x * ppc + t;
      bool active = (t < ppc) && (e < cnt);
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
      tc_rounds<OBJ>(o, sm, t, ppc / TC_GROUP, load, finish);
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

// Hands Like Clouds on the tensor-core evaluator: point t of the tile = (sample t / M, draw t % M), M <= 128.
// the same as a call (QUAD form of k_hlc_tc: the kernel inlines load() several times -- prologue and loop of both operand
// forms -- and each copy of the generator is ~10 k instructions; as a function the kernel is a third of the size and its
// Hands-Like-Clouds step 8 % faster; the RFF form, with one copy, is faster inlined)
__device__ __noinline__ void hlc_normals_call(uint64_t seed, int i, int cycle, int iter, int k, int d, float (&u)[TC_D]) {
  hlc_normals(seed, i, cycle, iter, k, d, u);
}

// QUAD and RFF forms: a draw's normals are generated once, in load, and kept in shared memory for the reduction (row t
// of one of two buffers, by tile parity: the QUAD form fetches a tile's point two tiles ahead of its finish).  The
// x-stationary GMM_FULL form has no shared memory left for them (its W stages fill it): it regenerates them in finish --
// with fp16 operands k_hlc_tcx below takes its place.
struct HlcCtx { int i; bool valid; };
template <int OBJ>
__global__ void __launch_bounds__(TC_THREADS, 1) k_hlc_tc(const TcObj o, const HlcArgs a) {
  extern __shared__ __align__(1024) unsigned char tc_smem_raw[];
  const TcSmem sm = tc_carve(tc_smem_raw);
  const int t = threadIdx.x, d = a.d, M = a.M;
  const float sigma = *a.sigma_dev;
  if (sigma == 0.0f) return;                       // no spread among the unfrozen samples: nobody moves (R-18)
  const int spt = min(TC_PTS / M, HLC_MAX_SPT);
  const bool m_pow2 = (M & (M - 1)) == 0;              // f / M = f * (1 / M) exactly: the baseline's M divisions per item become multiplications
  const float inv_m = 1.0f / (float)M;
  const int cnt = a.count ? *a.count : a.max_count;
  const int ntiles = (cnt + spt - 1) / spt;
  if ((int)blockIdx.x >= ntiles) return;
  tc_begin<OBJ>(sm, t);
  const int s = t / M, k = t - s * M;
  constexpr bool KEEP_U = OBJ != CHISAO_OBJ_GMM_FULL;
  constexpr int US = (OBJ == CHISAO_OBJ_RFF) ? RFF_TC_D + 1 : TC_D + 1;      // row stride of the normals (conflict-free)
  // buffer 0 in the kernel scratch; buffer 1 behind it (RFF: 2 x 33 KB fit the scratch) or behind the resident QUAD record
  float *Us0 = reinterpret_cast<float *>(sm.scratch());
  float *Us1 = (OBJ == CHISAO_OBJ_RFF) ? Us0 + TC_PTS * US
                                       : reinterpret_cast<float *>(sm.scratch() + TC_SCRATCH_BYTES + ((TC_REC_BYTES + 255) & ~255));
  static_assert(2 * TC_PTS * (RFF_TC_D + 1) * 4 <= TC_SCRATCH_BYTES, "RFF: two normals buffers in the scratch");
  static_assert(TC_PTS * (TC_D + 1) * 4 <= TC_SCRATCH_BYTES && ((TC_REC_BYTES + 255) & ~255) + TC_PTS * (TC_D + 1) * 4 <= 2 * TCX_W_BYTES, "QUAD: normals buffers");
  auto ubuf = [&](int tile) { return ((((tile - (int)blockIdx.x) / (int)gridDim.x) & 1) && KEEP_U) ? Us1 : Us0; };
  auto load = [&](int tile, float (&x)[TC_D]) -> HlcCtx {
    HlcCtx c;
    const int first = tile * spt;
    c.valid = (s < spt) && (first + s < cnt);
    c.i = c.valid ? a.list[first + s] : 0;
    if (c.valid) {
      float u[TC_D];
      if constexpr (OBJ == CHISAO_OBJ_QUAD) hlc_normals_call(a.seed, c.i, a.cycle, a.iter, k, d, u);
      else hlc_normals(a.seed, c.i, a.cycle, a.iter, k, d, u);
      if constexpr (KEEP_U) {
        float *row = ubuf(tile) + t * US;
#pragma unroll
        for (int q = 0; q < US - 1; ++q) row[q] = u[q];
      }
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
    float *Us = ubuf(tile);
    float *fvs = sm.fvs();                                      // [256] values
    if constexpr (!KEEP_U) compute_sync();                      // the previous tile's estimate has been read out of the scratch
    if (c.valid) {
      val += eval_noise(o.sigma_noise, a.seed, a.cycle, i, 5, a.iter, k);
      a.hlc_f[(size_t)i * M + k] = val;
      if constexpr (!KEEP_U) {
        float u[TC_D];
        hlc_normals(a.seed, i, a.cycle, a.iter, k, d, u);
#pragma unroll
        for (int q = 0; q < TC_D; ++q) Us[t * US + q] = u[q];
      }
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
      if (a.baseline) for (int kk = 0; kk < M; ++kk) b += m_pow2 ? fvs[ss * M + kk] * inv_m : fvs[ss * M + kk] / (float)M;
      float acc = 0.0f;
      for (int kk = 0; kk < M; ++kk) acc = fmaf(fvs[ss * M + kk] - b, Us[(ss * M + kk) * US + j], acc);
      const float gh = acc / ((float)M * sigma);
      a.ghat[(size_t)ii * d + j] = gh;
      const float xo = a.x[(size_t)ii * d + j];
      a.x[(size_t)ii * d + j] = clipf(fmaf(a.eta, gh, xo), a.lo[j], a.hi[j]);
    }
    if constexpr (KEEP_U) compute_sync();                       // everybody has read fvs and this buffer: the next loads may overwrite them
    if (t == 0) atomicAdd(&a.evals[EV_HLC], (unsigned long long)nval * (unsigned long long)M);
  };
  tc_run<OBJ>(o, sm, t, ntiles, load, finish);
  tc_teardown(sm, t);
}

// ---- Hands Like Clouds, GMM_FULL with fp16 operands: normals generated ONCE, by warps of their own ---------------------
// k_hlc_tc above generates the d normals of a draw twice (for the evaluation point and again for the reduction), on
// the warps that drain the accumulators, while the tensor pipe waits: at C5 the kernel ran at 0.45 of the FD kernel's
// evaluation rate.  Here four more warps (10..13; warp w owns TMEM lanes 32 (w & 3) .. + 31 of both groups) generate
// the normals of the NEXT tile under the current tile's MMAs: they keep u in shared memory for the reduction
// (two tiles of 256 x 64 fp32, XOR-swizzled 16-byte chunks), form x + sigma u, split it into fp16 hi / lo and write
// the X image of their 32 points straight into TMEM.  The compute warps only drain (tcx_compute<EXT>), add the noise and
// reduce.  Barriers: xfree(g) "the group's last MMAs of the tile retired" (compute -> generators), xbar(g) "X image
// written" (generators -> issuer), ufull(b) / ufree(b) for the two normals buffers.
constexpr int HLCX_THREADS = TC_THREADS + 128;
__device__ __forceinline__ float *hlcx_u_chunk(const TcSmem &sm, int buf, int pt, int c4) {   // 16-byte chunk c4 of point pt
  return reinterpret_cast<float *>(sm.scratch() + (size_t)buf * HLCX_U_BYTES + (size_t)pt * (TC_D * 4) + (size_t)((c4 ^ (pt & 15)) * 16));
}
// Software pipeline of a generator warp over the CTA's tiles:  A(0);  for it: B(it); A(it + 1)
//   A(it): the normals of tile `it` -> normals buffer it & 1 (after the reduction of tile it - 2 has read it), and the
//          centre rows of the tile's samples -> shared memory;  this is the expensive part (Philox + Box-Muller, ~70
//          instructions per normal) and runs under the MMAs of tile it - 1
//   B(it): after the group's last MMAs of tile it - 1 have retired: x + sigma u from shared memory, fp16 hi / lo split,
//          tcgen05.st into the X image, "image written" -- a few hundred instructions on the tensor pipe's critical path
__device__ __forceinline__ void gen_sync() { asm volatile("bar.sync 5, 128;" ::: "memory"); }   // the four generator warps
__device__ __forceinline__ void hlcx_generator(const TcObj &o, const TcSmem &sm, const HlcArgs &a, int t, int ntc, int cnt, int spt, float sigma) {
  const uint32_t tm = *sm.tmem();
  const int lane = t & 31, q = (t >> 5) & 3, d = a.d, M = a.M;
  const int gt = q * 32 + lane;                                    // index among the 128 generator threads
  const uint32_t lanes = tm + ((uint32_t)(q * 32) << 16);
  {   // the constant operand row (1, 1, 1, 0, ...) of the -c step: columns [64, 80) of both groups, once
    uint32_t one[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) one[c] = 0u;
    one[0] = 0x3C003C00u; one[1] = 0x00003C00u;
    tc_st16u(lanes + 64, one);
    tc_st16u(lanes + 256 + 64, one);
  }
  const uint32_t tg = rng_tag(5, a.iter, PUR_HLC_U);
  float4 *xr4 = reinterpret_cast<float4 *>(sm.xrows());
  auto phase_a = [&](int it) {
    const int tile = (int)blockIdx.x + it * (int)gridDim.x, first = tile * spt, buf = it & 1;
    if (it >= 2) mbar_wait(sm.ufree(buf), ((it >> 1) - 1) & 1);    // the reduction of tile it - 2 has read this buffer
    // centre rows of the tile's samples (zero beyond the list and beyond d): [spt][16] float4
    for (int e = gt; e < spt * (TC_D / 4); e += 128) {
      const int sr = e >> 4, c4 = e & 15;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (first + sr < cnt && 4 * c4 < d) v = *reinterpret_cast<const float4 *>(a.x + (size_t)a.list[first + sr] * d + 4 * c4);
      xr4[e] = v;
    }
#pragma unroll 1
    for (int g = 0; g < 2; ++g) {
      const int pt = g * TC_GROUP + q * 32 + lane;
      const int s = pt / M, k = pt - s * M;
      const bool valid = (s < spt) && (first + s < cnt);
      const int i = valid ? a.list[first + s] : 0;
      const uint32_t b0 = ((uint32_t)k * (uint32_t)d) >> 2;        // first Philox block of the draw (d is a multiple of 4)
#pragma unroll 4
      for (int c4 = 0; c4 < TC_D / 4; ++c4) {
        float4 u = make_float4(0.f, 0.f, 0.f, 0.f);
        if (valid && 4 * c4 < d && !TC_EXP(o, 2)) {
          const uint4 w = philox_block(a.seed, b0 + (uint32_t)c4, (uint32_t)i, (uint32_t)a.cycle, tg);
          box_muller(w.x, w.y, u.x, u.y);
          box_muller(w.z, w.w, u.z, u.w);
        }
        *reinterpret_cast<float4 *>(hlcx_u_chunk(sm, buf, pt, c4)) = u;
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.ufull(buf));                     // (mbarrier.arrive has release semantics: the stores above are visible to the waiters)
    gen_sync();                                                    // the centre rows are complete
  };
  auto phase_b = [&](int it) {
    const int buf = it & 1;
#pragma unroll 1
    for (int g = 0; g < 2; ++g) {
      const int pt = g * TC_GROUP + q * 32 + lane;
      const int s = min(pt / M, HLC_MAX_SPT - 1);                  // (rows of idle points are zero like their normals)
      const uint32_t xaddr = lanes + (uint32_t)(g * 256);
      if (it >= 1) mbar_wait(sm.xfree(g), (it - 1) & 1);            // the group's MMAs of the previous tile are done with the image
      asm volatile("tcgen05.fence::after_thread_sync;");
#pragma unroll
      for (int hq = 0; hq < 2; ++hq) {                             // coordinates 32 hq .. 32 hq + 31
        uint32_t h[16], l[16];
#pragma unroll
        for (int b = 0; b < 8; ++b) {
          const int c4 = 8 * hq + b;
          const float4 u = *reinterpret_cast<const float4 *>(hlcx_u_chunk(sm, buf, pt, c4));
          const float4 xv = (pt / M < spt) ? xr4[s * (TC_D / 4) + c4] : make_float4(0.f, 0.f, 0.f, 0.f);
          const float x0 = fmaf(sigma, u.x, xv.x), x1 = fmaf(sigma, u.y, xv.y), x2 = fmaf(sigma, u.z, xv.z), x3 = fmaf(sigma, u.w, xv.w);
          const __half h0 = __float2half_rn(x0), h1 = __float2half_rn(x1), h2 = __float2half_rn(x2), h3 = __float2half_rn(x3);
          const __half l0 = __float2half_rn(x0 - __half2float(h0)), l1 = __float2half_rn(x1 - __half2float(h1));
          const __half l2 = __float2half_rn(x2 - __half2float(h2)), l3 = __float2half_rn(x3 - __half2float(h3));
          h[2 * b] = (uint32_t)__half_as_ushort(h0) | ((uint32_t)__half_as_ushort(h1) << 16);
          h[2 * b + 1] = (uint32_t)__half_as_ushort(h2) | ((uint32_t)__half_as_ushort(h3) << 16);
          l[2 * b] = (uint32_t)__half_as_ushort(l0) | ((uint32_t)__half_as_ushort(l1) << 16);
          l[2 * b + 1] = (uint32_t)__half_as_ushort(l2) | ((uint32_t)__half_as_ushort(l3) << 16);
        }
        tc_st16u(xaddr + 16 * hq, h);
        tc_st16u(xaddr + 32 + 16 * hq, l);
      }
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      asm volatile("tcgen05.fence::before_thread_sync;");
      __syncwarp();
      if (lane == 0) mbar_arrive(sm.xbar(g));
    }
    gen_sync();                                                    // every warp is done with the centre rows: A(it + 1) may overwrite them
  };
  phase_a(0);
  for (int it = 0; it < ntc; ++it) {
    phase_b(it);
    if (it + 1 < ntc) phase_a(it + 1);
  }
}

__global__ void __launch_bounds__(HLCX_THREADS, 1) k_hlc_tcx(const TcObj o, const HlcArgs a) {
  extern __shared__ __align__(1024) unsigned char tc_smem_raw[];
  const TcSmem sm = tc_carve(tc_smem_raw);
  const int t = threadIdx.x, d = a.d, M = a.M;
  const float sigma = *a.sigma_dev;
  if (sigma == 0.0f) return;                       // no spread among the unfrozen samples: nobody moves (R-18)
  const int spt = min(TC_PTS / M, HLC_MAX_SPT);
  const bool m_pow2 = (M & (M - 1)) == 0;              // f / M = f * (1 / M) exactly: the baseline's M divisions per item become multiplications
  const float inv_m = 1.0f / (float)M;
  const int cnt = a.count ? *a.count : a.max_count;
  const int ntiles = (cnt + spt - 1) / spt;
  if ((int)blockIdx.x >= ntiles) return;
  tc_setup(sm, t, 1);
  const int ntc = tcx_tiles_of_cta(ntiles);
  const int warp = __shfl_sync(0xffffffffu, t >> 5, 0);   // provably warp-uniform role index
  if (warp < TC_PTS / 32) {
    const int s = t / M, k = t - s * M;
    float *fvs = sm.fvs();
    auto noload = [](int, float (&)[1]) -> int { return 0; };
    // Positions are only written by the tile that owns the sample; the generators read the NEXT tile's (other) samples.
    auto finish = [&](int tile, float val, int it) {
      const int first = tile * spt, buf = it & 1;
      const bool valid = (s < spt) && (first + s < cnt);
      const int i = valid ? a.list[first + s] : 0;
      compute_sync();                        // the previous tile's reduction has read fvs
      if (valid) {
        val += eval_noise(o.sigma_noise, a.seed, a.cycle, i, 5, a.iter, k);
        a.hlc_f[(size_t)i * M + k] = val;
      } else {
        val = 0.f;
      }
      fvs[t] = val;
      mbar_wait(sm.ufull(buf), (it >> 1) & 1);   // the tile's normals are in shared memory
      compute_sync();
      const int nval = TC_EXP(o, 4) ? 0 : min(spt, cnt - first);
      for (int item = t; item < nval * d; item += TC_PTS) {
        const int ss = item / d, j = item - ss * d;
        const int ii = a.list[first + ss];
        float b = 0.0f;
        if (a.baseline) for (int kk = 0; kk < M; ++kk) b += m_pow2 ? fvs[ss * M + kk] * inv_m : fvs[ss * M + kk] / (float)M;
        float acc = 0.0f;
        for (int kk = 0; kk < M; ++kk) acc = fmaf(fvs[ss * M + kk] - b, hlcx_u_chunk(sm, buf, ss * M + kk, j >> 2)[j & 3], acc);
        const float gh = acc / ((float)M * sigma);
        a.ghat[(size_t)ii * d + j] = gh;
        const float xo = a.x[(size_t)ii * d + j];
        a.x[(size_t)ii * d + j] = clipf(fmaf(a.eta, gh, xo), a.lo[j], a.hi[j]);
      }
      __syncwarp();
      if ((t & 31) == 0) mbar_arrive(sm.ufree(buf));
      if (t == 0) atomicAdd(&a.evals[EV_HLC], (unsigned long long)nval * (unsigned long long)M);
    };
    tcx_compute<true>(o, sm, t, ntc, noload, finish);
  } else if (warp == TC_PTS / 32) {
    if (t == TC_PTS) tcx_loader(o, sm, ntc, 2, HLCX_W_OFF);
  } else if (warp == TC_PTS / 32 + 1) {
    tcx_issuer(o, sm, ntc, 2, HLCX_W_OFF);
  } else {
    hlcx_generator(o, sm, a, t, ntc, cnt, spt, sigma);
  }
  tc_teardown(sm, t);
}

// ---- launchers ------------------------------------------------------------------------------------------------
static int g_tc_sms = 148;
static int g_exp = 0;
static bool g_hlc_plain = false;   // CHISAO_HLC_PLAIN in the environment: keep k_hlc_tc for GMM_FULL (A/B measurements)
static inline int tc_grid(int obj_id, int ntiles) {   // persistent CTAs, one per SM
  (void)obj_id;
  return ntiles > g_tc_sms ? g_tc_sms : ntiles;
}
cudaError_t tc_configure() {
  cudaError_t e;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
    g_tc_sms = sms;
  g_hlc_plain = getenv("CHISAO_HLC_PLAIN") != nullptr;
  g_exp = getenv("CHISAO_EXP") ? atoi(getenv("CHISAO_EXP")) : 0;
#define CFG(K) if ((e = cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM_BYTES)) != cudaSuccess) return e;
  CFG(k_eval_fd_tc<CHISAO_OBJ_GMM_FULL>) CFG(k_eval_fd_tc<CHISAO_OBJ_QUAD>)
  CFG(k_eval_points_tc<CHISAO_OBJ_GMM_FULL>) CFG(k_eval_points_tc<CHISAO_OBJ_QUAD>)
  CFG(k_hlc_tc<CHISAO_OBJ_GMM_FULL>) CFG(k_hlc_tc<CHISAO_OBJ_QUAD>)
  CFG(k_eval_fd_tc<CHISAO_OBJ_RFF>) CFG(k_eval_points_tc<CHISAO_OBJ_RFF>) CFG(k_hlc_tc<CHISAO_OBJ_RFF>)
  CFG(k_hlc_tcx)
#undef CFG
  return cudaSuccess;
}
cudaError_t launch_fd_tc(int obj_id, const TcObj &o_in, const FdArgs &a, int n_samples, cudaStream_t st) {
  TcObj o = o_in; o.exp = g_exp;
  const int spt = fd_tc_samples_per_tile(a.d);
  const int grid = tc_grid(obj_id, (n_samples + spt - 1) / spt);
  if (obj_id == CHISAO_OBJ_QUAD) k_eval_fd_tc<CHISAO_OBJ_QUAD><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else if (obj_id == CHISAO_OBJ_RFF) k_eval_fd_tc<CHISAO_OBJ_RFF><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else k_eval_fd_tc<CHISAO_OBJ_GMM_FULL><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  return cudaGetLastError();
}
cudaError_t launch_pt_tc(int obj_id, const TcObj &o_in, const PtArgs &a_in, int n_samples, cudaStream_t st) {
  TcObj o = o_in; o.exp = g_exp;
  PtArgs a = a_in;
  // tile-local rounds: one tile per CTA; a worklist that would fill fewer CTAs than there are SMs is cut into tiles of
  // one group (128 entries): every round of a tile costs a full tile evaluation, and half-size tiles on twice the SMs halve it
  a.tc_pts = (a.mode == PT_LS_ALL && obj_id != CHISAO_OBJ_GMM_FULL && (n_samples + TC_PTS - 1) / TC_PTS < g_tc_sms) ? TC_GROUP : TC_PTS;
  const int ntiles = (n_samples + a.tc_pts - 1) / a.tc_pts;
  const int grid = (a.mode == PT_LS_ALL) ? ntiles : tc_grid(obj_id, (n_samples + TC_PTS - 1) / TC_PTS);
  if (obj_id == CHISAO_OBJ_QUAD) k_eval_points_tc<CHISAO_OBJ_QUAD><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else if (obj_id == CHISAO_OBJ_RFF) k_eval_points_tc<CHISAO_OBJ_RFF><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else k_eval_points_tc<CHISAO_OBJ_GMM_FULL><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  return cudaGetLastError();
}
cudaError_t launch_hlc_tc(int obj_id, const TcObj &o_in, const HlcArgs &a, int n_samples, cudaStream_t st) {
  TcObj o = o_in; o.exp = g_exp;
  const int spt = TC_PTS / a.M < HLC_MAX_SPT ? TC_PTS / a.M : HLC_MAX_SPT;
  const int grid = tc_grid(obj_id, (n_samples + spt - 1) / spt);
  if (obj_id == CHISAO_OBJ_QUAD) k_hlc_tc<CHISAO_OBJ_QUAD><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else if (obj_id == CHISAO_OBJ_RFF) k_hlc_tc<CHISAO_OBJ_RFF><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  else if (o.f16 && (a.d & 3) == 0 && !g_hlc_plain) k_hlc_tcx<<<grid, HLCX_THREADS, TC_SMEM_BYTES, st>>>(o, a);   // normals generated once, by warps of their own
  else k_hlc_tc<CHISAO_OBJ_GMM_FULL><<<grid, TC_THREADS, TC_SMEM_BYTES, st>>>(o, a);
  return cudaGetLastError();
}

}  // namespace chisao
