// chisao_eval.cuh -- the value-only objective evaluator ("accessible through evaluations
// f(theta)") and the three kernels built on it:
//   k_eval_fd     : 2d central-difference stencil points per sample -> g   (R-1)
//                   FD_ANTI additionally applies Eq. 6 in the epilogue
//   k_eval_points : one point per sample (cycle-start centre value, line-search trials; R-4)
//   k_hlc         : M Gaussian-perturbed points per sample -> smoothed-gradient step (PAPER.md:113-120,
//                   Eq. 9; north_star (e); R-11)
//
// Mapping: a CTA of NT = 128 threads evaluates a tile of PTILE = 256 points, two per thread (register
// tile: every parameter value fetched from shared memory feeds two FMA chains per row).  Points are staged
// in shared memory as float4 columns [DP/4][PTILE] (conflict-free LDS.128); objective parameters are
// streamed through shared memory in chunks of `kc` component records by the bulk-copy (TMA) engine with an
// mbarrier, double-buffered when the objective does not fit one chunk (GMM_FULL at d = 64: 1 MB).
// Every point is evaluated independently (black-box cost; no stencil sharing, see DESIGN.md NEXT-5).
#pragma once
#include "chisao_device.cuh"

namespace chisao {

// shared-memory carve of the evaluation kernels (dynamic):
//   [0, 16)            two mbarriers
//   [16, 16 + 2*CH)    parameter chunk buffers (CH = chunk bytes rounded to 16)
//   then               point columns float4[DP/4][PTILE]
//   then               kernel-specific scratch
struct EvalSmem {
  uint64_t *bar;
  float *chunk[2];
  float4 *pts;
  float *extra;
};
template <int DP>
__device__ __forceinline__ EvalSmem carve_smem(unsigned char *base, int chunk_floats) {
  EvalSmem s;
  s.bar = reinterpret_cast<uint64_t *>(base);
  s.chunk[0] = reinterpret_cast<float *>(base + 16);
  s.chunk[1] = s.chunk[0] + chunk_floats;
  s.pts = reinterpret_cast<float4 *>(s.chunk[1] + chunk_floats);
  s.extra = reinterpret_cast<float *>(s.pts + (DP / 4) * PTILE);
  return s;
}
inline size_t eval_smem_bytes(const DevObj &o, size_t extra_bytes) {
  const size_t chunk = (size_t)o.kc * o.rec * 4;
  const int nchunks = (o.K + o.kc - 1) / o.kc;
  return 16 + (nchunks > 1 ? 2 : 2) * chunk + (size_t)(o.DP / 4) * PTILE * 16 + extra_bytes;
}

// thread t owns the points in columns t and NT + t
__device__ __forceinline__ float4 ld_pt(const float4 *pts, int c4, int col) { return pts[c4 * PTILE + col]; }

// ---- per-record accumulation -----------------------------------------------------------------------
// running state per point: GMM -> (m, s) online log-sum-exp; RFF -> s = sum; QUAD -> s = q
template <int OBJ, int DP>
__device__ __forceinline__ void accum_records(const float *__restrict__ buf, int nrec, int rec, const float4 *pts,
                                              int t, float s0, float (&m)[PPT], float (&s)[PPT]) {
  if constexpr (OBJ == CHISAO_OBJ_RFF) {
    // t_j = w_j . x + b_j is accumulated in fp64 (B200 issues DFMA at half the FFMA rate): with |t| up to ~50
    // an fp32 running sum loses ~1e-5 in t, which the cosine passes on to f.  w is stored as doubles in the
    // record, x is promoted once per point; the reduced angle goes to the fp32 hardware cosine.
    constexpr int PG = (DP <= 32) ? PPT : 1;   // points held in registers at once
#pragma unroll
    for (int p0 = 0; p0 < PPT; p0 += PG) {
      double xp[PG][DP];
#pragma unroll
      for (int pp = 0; pp < PG; ++pp)
#pragma unroll
        for (int c4 = 0; c4 < DP / 4; ++c4) {
          const float4 v = ld_pt(pts, c4, (p0 + pp) * NT + t);
          xp[pp][4 * c4] = (double)v.x; xp[pp][4 * c4 + 1] = (double)v.y;
          xp[pp][4 * c4 + 2] = (double)v.z; xp[pp][4 * c4 + 3] = (double)v.w;
        }
      double sd[PG];
#pragma unroll
      for (int pp = 0; pp < PG; ++pp) sd[pp] = 0.0;
      for (int k = 0; k < nrec; ++k) {
        const double2 *w2 = reinterpret_cast<const double2 *>(buf + (size_t)k * rec);
        const float4 tail = *reinterpret_cast<const float4 *>(buf + (size_t)k * rec + 2 * DP);
        double acc[PG];
#pragma unroll
        for (int pp = 0; pp < PG; ++pp) acc[pp] = (double)tail.y;
#pragma unroll
        for (int c2 = 0; c2 < DP / 2; ++c2) {
          const double2 w = w2[c2];
#pragma unroll
          for (int pp = 0; pp < PG; ++pp) {
            acc[pp] = fma(w.x, xp[pp][2 * c2], acc[pp]);
            acc[pp] = fma(w.y, xp[pp][2 * c2 + 1], acc[pp]);
          }
        }
#pragma unroll
        for (int pp = 0; pp < PG; ++pp) {
          const double kq = rint(acc[pp] * 0.15915494309189535);
          const float red = (float)fma(-kq, 6.283185307179586, acc[pp]);
          sd[pp] += (double)(tail.x * __cosf(red));
        }
      }
#pragma unroll
      for (int pp = 0; pp < PG; ++pp) s[p0 + pp] += (float)sd[pp];
    }
  } else if constexpr (OBJ == CHISAO_OBJ_GMM_ISO || OBJ == CHISAO_OBJ_GMM_DIAG) {
    // the point stays in registers across all records
    float xp[PPT][DP];
#pragma unroll
    for (int pp = 0; pp < PPT; ++pp)
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        const float4 v = ld_pt(pts, c4, pp * NT + t);
        xp[pp][4 * c4] = v.x; xp[pp][4 * c4 + 1] = v.y; xp[pp][4 * c4 + 2] = v.z; xp[pp][4 * c4 + 3] = v.w;
      }
    for (int k = 0; k < nrec; ++k) {
      const float4 *r4 = reinterpret_cast<const float4 *>(buf + (size_t)k * rec);
      float acc[PPT];
#pragma unroll
      for (int pp = 0; pp < PPT; ++pp) acc[pp] = 0.0f;
      if constexpr (OBJ == CHISAO_OBJ_GMM_ISO) {
#pragma unroll
        for (int c4 = 0; c4 < DP / 4; ++c4) {
          const float4 mu = r4[c4];
#pragma unroll
          for (int pp = 0; pp < PPT; ++pp) {
            float e;
            e = xp[pp][4 * c4] - mu.x; acc[pp] = fmaf(e, e, acc[pp]);
            e = xp[pp][4 * c4 + 1] - mu.y; acc[pp] = fmaf(e, e, acc[pp]);
            e = xp[pp][4 * c4 + 2] - mu.z; acc[pp] = fmaf(e, e, acc[pp]);
            e = xp[pp][4 * c4 + 3] - mu.w; acc[pp] = fmaf(e, e, acc[pp]);
          }
        }
      } else if constexpr (OBJ == CHISAO_OBJ_GMM_DIAG) {
#pragma unroll
        for (int c4 = 0; c4 < DP / 4; ++c4) {
          const float4 mu = r4[c4], iv = r4[DP / 4 + c4];
#pragma unroll
          for (int pp = 0; pp < PPT; ++pp) {
            float e;
            e = (xp[pp][4 * c4] - mu.x) * iv.x; acc[pp] = fmaf(e, e, acc[pp]);
            e = (xp[pp][4 * c4 + 1] - mu.y) * iv.y; acc[pp] = fmaf(e, e, acc[pp]);
            e = (xp[pp][4 * c4 + 2] - mu.z) * iv.z; acc[pp] = fmaf(e, e, acc[pp]);
            e = (xp[pp][4 * c4 + 3] - mu.w) * iv.w; acc[pp] = fmaf(e, e, acc[pp]);
          }
        }
      }
      const float4 tail = (OBJ == CHISAO_OBJ_GMM_DIAG) ? r4[2 * (DP / 4)] : r4[DP / 4];
#pragma unroll
      for (int pp = 0; pp < PPT; ++pp) {
        {
          const float v = (OBJ == CHISAO_OBJ_GMM_ISO) ? fmaf(-acc[pp], s0, tail.x) : fmaf(-0.5f, acc[pp], tail.x);
          const float mn = fmaxf(m[pp], v);
          if (mn > -INFINITY) {   // online log-sum-exp
            s[pp] = s[pp] * __expf(m[pp] - mn) + __expf(v - mn);
            m[pp] = mn;
          }
        }
      }
    }
  } else {
    // GMM_FULL / QUAD: q = || W (x - mu) ||^2 accumulated over non-negative terms
    constexpr int RB = 4;  // rows per register block
    for (int k = 0; k < nrec; ++k) {
      const float *rbase = buf + (size_t)k * rec;
      const float4 *W4 = reinterpret_cast<const float4 *>(rbase);
      const float4 *mu4 = reinterpret_cast<const float4 *>(rbase + DP * DP);
      float df[PPT][DP];
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        const float4 mu = mu4[c4];
#pragma unroll
        for (int pp = 0; pp < PPT; ++pp) {
          const float4 v = ld_pt(pts, c4, pp * NT + t);
          df[pp][4 * c4] = v.x - mu.x; df[pp][4 * c4 + 1] = v.y - mu.y;
          df[pp][4 * c4 + 2] = v.z - mu.z; df[pp][4 * c4 + 3] = v.w - mu.w;
        }
      }
      float q[PPT];
#pragma unroll
      for (int pp = 0; pp < PPT; ++pp) q[pp] = 0.0f;
#pragma unroll 1
      for (int r = 0; r < DP; r += RB) {
        float z[PPT][RB];
#pragma unroll
        for (int pp = 0; pp < PPT; ++pp)
#pragma unroll
          for (int rb = 0; rb < RB; ++rb) z[pp][rb] = 0.0f;
#pragma unroll
        for (int c4 = 0; c4 < DP / 4; ++c4) {
          float4 w[RB];
#pragma unroll
          for (int rb = 0; rb < RB; ++rb) w[rb] = W4[(r + rb) * (DP / 4) + c4];
#pragma unroll
          for (int pp = 0; pp < PPT; ++pp)
#pragma unroll
            for (int rb = 0; rb < RB; ++rb) {
              z[pp][rb] = fmaf(w[rb].x, df[pp][4 * c4], z[pp][rb]);
              z[pp][rb] = fmaf(w[rb].y, df[pp][4 * c4 + 1], z[pp][rb]);
              z[pp][rb] = fmaf(w[rb].z, df[pp][4 * c4 + 2], z[pp][rb]);
              z[pp][rb] = fmaf(w[rb].w, df[pp][4 * c4 + 3], z[pp][rb]);
            }
        }
#pragma unroll
        for (int pp = 0; pp < PPT; ++pp)
#pragma unroll
          for (int rb = 0; rb < RB; ++rb) q[pp] = fmaf(z[pp][rb], z[pp][rb], q[pp]);
      }
      const float a = rbase[DP * DP + DP];
#pragma unroll
      for (int pp = 0; pp < PPT; ++pp) {
        if constexpr (OBJ == CHISAO_OBJ_QUAD) {
          s[pp] += q[pp];
        } else {
          const float v = fmaf(-0.5f, q[pp], a);
          const float mn = fmaxf(m[pp], v);
          if (mn > -INFINITY) {
            s[pp] = s[pp] * __expf(m[pp] - mn) + __expf(v - mn);
            m[pp] = mn;
          }
        }
      }
    }
  }
}

// ---- Appendix-D benchmark functions, negated for maximisation ----------------------
// One staged point (column `col`), function chosen by the objective id (uniform over the launch).  The sums are
// rearranged so that no large constant is cancelled in fp32 (the rearrangements are exact identities):
//   Rastrigin  10 d + sum (x^2 - 10 cos 2 pi x)        = sum (x^2 + 20 sin^2(pi x))
//   Ackley     -20 e^{-0.2 r} - e^{c} + 20 + e          = -20 expm1(-0.2 r) - e expm1(c - 1),
//              c - 1 = (1/d) sum (cos 2 pi x - 1)       = -(2/d) sum sin^2(pi x)
// sin(pi x) uses sinpif (exact argument reduction).  Where fp32 cannot deliver the 1e-5 bar on f, the critical
// sub-expression runs in fp64 (B200 issues DFMA at half the FFMA rate): Schwefel's x sin(sqrt|x|) near x = 421
// (418.98 - 418.98 at the optimum), Michalewicz's angle i x^2 / pi (up to 200 rad under a 20th power), Trid's
// O(d^4) products that cancel to O(d^3), Styblinski-Tang's mixed-sign polynomial terms, and Bukin's ridge distance y - 0.01 x^2 under a square root.
template <int DP>
__device__ __forceinline__ float appd_point(int id, int d, const float4 *pts, int col) {
  float x[DP];
#pragma unroll
  for (int c4 = 0; c4 < DP / 4; ++c4) {
    const float4 v = ld_pt(pts, c4, col);
    x[4 * c4] = v.x; x[4 * c4 + 1] = v.y; x[4 * c4 + 2] = v.z; x[4 * c4 + 3] = v.w;
  }
  switch (id) {
    case CHISAO_OBJ_RASTRIGIN: {
      float acc = 0.0f;
#pragma unroll
      for (int j = 0; j < DP; ++j)
        if (j < d) { const float sp = sinpif(x[j]); acc = fmaf(x[j], x[j], acc); acc = fmaf(20.0f * sp, sp, acc); }
      return -acc;
    }
    case CHISAO_OBJ_ACKLEY: {
      float s2 = 0.0f, ss = 0.0f;
#pragma unroll
      for (int j = 0; j < DP; ++j)
        if (j < d) { const float sp = sinpif(x[j]); s2 = fmaf(x[j], x[j], s2); ss = fmaf(sp, sp, ss); }
      const float inv_d = 1.0f / (float)d;
      return 20.0f * expm1f(-0.2f * sqrtf(s2 * inv_d)) + 2.7182818284590452f * expm1f(-2.0f * ss * inv_d);
    }
    case CHISAO_OBJ_SCHWEFEL: {
      // rolled loop straight from shared memory (the fp64 sine dominates); sin(a) = sinpi(a / pi), a <= 22.4
      const float *pf = reinterpret_cast<const float *>(pts + col);
      double acc = 0.0;
#pragma unroll 2
      for (int j = 0; j < d; ++j) {
        const double t = (double)pf[(j >> 2) * (PTILE * 4) + (j & 3)];
        acc += 418.9829 - t * sinpi(sqrt(fabs(t)) * 0.3183098861837907);
      }
      return (float)(-acc);
    }
    case CHISAO_OBJ_STYBLINSKI_TANG: {
      double acc = 0.0;   // terms of either sign up to 80 cancel across coordinates: three DFMA per coordinate
#pragma unroll
      for (int j = 0; j < DP; ++j)
        if (j < d) { const double t = (double)x[j], t2 = t * t; acc += fma(t2, t2 - 16.0, 5.0 * t); }
      return (float)(-0.5 * acc);
    }
    case CHISAO_OBJ_MICHALEWICZ: {
      float acc = 0.0f;
#pragma unroll
      for (int j = 0; j < DP; ++j)
        if (j < d) {
          const double t = (double)x[j];
          const double turns = (double)(j + 1) * t * t * 0.10132118364233778;   // angle / pi = i x^2 / pi^2
          const float fr = (float)(turns - 2.0 * rint(0.5 * turns));            // angle / pi reduced to [-1, 1]
          const float sa = sinpif(fr), s2 = sa * sa, s4 = s2 * s2, s8 = s4 * s4, s16 = s8 * s8;
          acc = fmaf(sinpif(x[j] * 0.31830988618f), s16 * s4, acc);   // sin(x), x in [0, pi]: no slow-path reduction
        }
      return acc;
    }
    case CHISAO_OBJ_TRID: {
      double acc = 0.0, prev = 0.0;
#pragma unroll
      for (int j = 0; j < DP; ++j)
        if (j < d) { const double t = (double)x[j]; acc = fma(t - 1.0, t - 1.0, acc); acc = fma(-t, prev, acc); prev = t; }
      return (float)(-acc);
    }
    default: {  // CHISAO_OBJ_BUKIN6 (d = 2)
      const double u = (double)x[1] - 0.01 * (double)x[0] * (double)x[0];
      return -(100.0f * sqrtf((float)fabs(u)) + 0.01f * fabsf(x[0] + 10.0f));
    }
  }
}

// Evaluate the thread's PPT staged points.  Must be called by every thread of the CTA (contains barriers);
// the points must already be visible in shared memory (caller syncs).  `use` counts bulk copies issued on
// each mbarrier so far (phase tracking when a kernel evaluates more than one tile).
template <int OBJ, int DP>
__device__ __forceinline__ void eval_tile(const DevObj &o, const EvalSmem &sm, int t, uint32_t &use, float (&fout)[PPT]) {
  if constexpr (OBJ == CHISAO_OBJ_APPD) {   // parameter-free: nothing to stream
#pragma unroll 1
    for (int pp = 0; pp < PPT; ++pp) fout[pp] = appd_point<DP>(o.id, o.d, sm.pts, pp * NT + t);
  } else {
  float m[PPT], s[PPT];
#pragma unroll
  for (int pp = 0; pp < PPT; ++pp) { m[pp] = -INFINITY; s[pp] = 0.0f; }
  const int nchunks = (o.K + o.kc - 1) / o.kc;
  const uint32_t chunk_floats = (uint32_t)o.kc * o.rec;
  if (nchunks == 1 && use != 0) {
    // the whole objective fits one chunk and an earlier call of this CTA has landed it in buffer 0: it is still there
    accum_records<OBJ, DP>(sm.chunk[0], o.K, o.rec, sm.pts, t, o.s0, m, s);
  } else {
  if (t == 0) {  // first chunk
    const int n0 = min(o.kc, o.K);
    mbar_expect_tx(&sm.bar[use & 1], (uint32_t)n0 * o.rec * 4);
    bulk_g2s(sm.chunk[use & 1], o.recs, (uint32_t)n0 * o.rec * 4, &sm.bar[use & 1]);
  }
  for (int c = 0; c < nchunks; ++c) {
    const uint32_t u = use + c;
    if (c + 1 < nchunks) {
      __syncthreads();  // every thread is done with the buffer chunk c+1 will overwrite
      if (t == 0) {
        const int n1 = min(o.kc, o.K - (c + 1) * o.kc);
        mbar_expect_tx(&sm.bar[(u + 1) & 1], (uint32_t)n1 * o.rec * 4);
        bulk_g2s(sm.chunk[(u + 1) & 1], o.recs + (size_t)(c + 1) * chunk_floats, (uint32_t)n1 * o.rec * 4,
                 &sm.bar[(u + 1) & 1]);
      }
    }
    mbar_wait(&sm.bar[u & 1], (u >> 1) & 1);
    const int nrec = min(o.kc, o.K - c * o.kc);
    accum_records<OBJ, DP>(sm.chunk[u & 1], nrec, o.rec, sm.pts, t, o.s0, m, s);
  }
  use += nchunks;
  }
#pragma unroll
  for (int pp = 0; pp < PPT; ++pp) {
    if constexpr (OBJ == CHISAO_OBJ_RFF) {
      // -s0 ||x||^2 + sum (the quadratic part from the staged point)
      float n2 = 0.0f;
#pragma unroll
      for (int c4 = 0; c4 < DP / 4; ++c4) {
        const float4 v = ld_pt(sm.pts, c4, pp * NT + t);
        n2 = fmaf(v.x, v.x, n2); n2 = fmaf(v.y, v.y, n2); n2 = fmaf(v.z, v.z, n2); n2 = fmaf(v.w, v.w, n2);
      }
      fout[pp] = fmaf(-o.s0, n2, s[pp]);
    } else if constexpr (OBJ == CHISAO_OBJ_QUAD) {
      fout[pp] = -0.5f * s[pp];
    } else {
      fout[pp] = m[pp] + logf(s[pp]);
    }
  }
  }
}

// row loader: coordinates 4*c4 .. 4*c4+3 of a [*][d] row, zero beyond d
__device__ __forceinline__ float4 ld_row4(const float *row, int c4, int d, bool vec) {
  if (vec) return (4 * c4 < d) ? *(reinterpret_cast<const float4 *>(row) + c4) : make_float4(0.f, 0.f, 0.f, 0.f);
  float4 v;
  v.x = (4 * c4 < d) ? row[4 * c4] : 0.0f;
  v.y = (4 * c4 + 1 < d) ? row[4 * c4 + 1] : 0.0f;
  v.z = (4 * c4 + 2 < d) ? row[4 * c4 + 2] : 0.0f;
  v.w = (4 * c4 + 3 < d) ? row[4 * c4 + 3] : 0.0f;
  return v;
}
__device__ __forceinline__ void set4(float4 &v, int l, float val) {
  if (l == 0) v.x = val; else if (l == 1) v.y = val; else if (l == 2) v.z = val; else v.w = val;
}
__device__ __forceinline__ float get4(const float4 &v, int l) { return l == 0 ? v.x : (l == 1 ? v.y : (l == 2 ? v.z : v.w)); }

}  // namespace chisao
