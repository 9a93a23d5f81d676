// chisao_device.cuh -- device helpers: counter-based randomness, warp reductions, small utilities.
#pragma once
#include "chisao_common.cuh"

namespace chisao {

// ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), R-15 ---------------------------
// counter = (c0 = block index in the draw sequence, c1 = sample / slot, c2 = cycle, c3 = tag),
// key = (seed_lo, seed_hi).  BASELINE.json north_star: "counter-based Philox stream keyed by
// (seed, cycle, sample, draw)".
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}
__device__ __forceinline__ uint4 philox_block(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
  return philox4x32_10(c0, c1, c2, c3, (uint32_t)seed, (uint32_t)(seed >> 32));
}
__host__ __device__ __forceinline__ uint32_t rng_tag(int phase, int iter, int purpose) {
  return ((uint32_t)phase << 24) | ((uint32_t)(iter & 0xFFFF) << 8) | (uint32_t)purpose;
}
// word -> uniform in (0,1): (2k+1)/2^24 with k = w >> 9 (23 bits), exact in fp32
__device__ __forceinline__ float u01(uint32_t w) { return ((float)(w >> 9) + 0.5f) * (1.0f / 8388608.0f); }

// Box-Muller on one pair of words: z0 = r cos(2 pi u2), z1 = r sin(2 pi u2), r = sqrt(-2 ln u1).
// sincospif(2 u2) keeps the angle exact (2 u2 is exact in fp32).
__device__ __forceinline__ void box_muller(uint32_t wa, uint32_t wb, float &z0, float &z1) {
  const float r = sqrtf(-2.0f * logf(u01(wa)));
  float sn, cs;
  sincospif(2.0f * u01(wb), &sn, &cs);
  z0 = r * cs; z1 = r * sn;
}
// n-th uniform / normal of the sequence (c1, c2, c3): word (n mod 4) of block (n div 4)
__device__ __forceinline__ float rng_uniform(uint64_t seed, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t n) {
  const uint4 w = philox_block(seed, n >> 2, c1, c2, c3);
  const uint32_t l = n & 3u;
  return u01(l == 0 ? w.x : (l == 1 ? w.y : (l == 2 ? w.z : w.w)));
}
__device__ __forceinline__ float rng_normal(uint64_t seed, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t n) {
  const uint4 w = philox_block(seed, n >> 2, c1, c2, c3);
  float z0, z1;
  if (n & 2u) box_muller(w.z, w.w, z0, z1); else box_muller(w.x, w.y, z0, z1);
  return (n & 1u) ? z1 : z0;
}
// additive evaluation noise, one draw per evaluation keyed structurally (R-2)
__device__ __forceinline__ float eval_noise(float sigma_noise, uint64_t seed, int cycle, int sample, int phase,
                                            int iter, int slot) {
  if (sigma_noise == 0.0f) return 0.0f;
  const uint4 w = philox_block(seed, (uint32_t)slot, (uint32_t)sample, (uint32_t)cycle, rng_tag(phase, iter, PUR_NOISE));
  float z0, z1;
  box_muller(w.x, w.y, z0, z1);
  return sigma_noise * z0;
}

// ---- warp reductions ------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ unsigned int warp_sum_u(unsigned int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

__device__ __forceinline__ float clipf(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }

// order-preserving map float -> uint32 (for atomicMax on f_max); 0 is below every image
__device__ __forceinline__ uint32_t enc_ordered(float f) {
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__host__ __device__ __forceinline__ float dec_ordered(uint32_t e) {
  if (e == 0u) {
#ifdef __CUDA_ARCH__
    return __uint_as_float(0xff800000u);
#else
    union { uint32_t u; float f; } c; c.u = 0xff800000u; return c.f;
#endif
  }
  const uint32_t u = (e & 0x80000000u) ? (e & 0x7fffffffu) : ~e;
#ifdef __CUDA_ARCH__
  return __uint_as_float(u);
#else
  union { uint32_t u; float f; } c; c.u = u; return c.f;
#endif
}

// ---- mbarrier + 1-D bulk copy (TMA engine, SASS UBLKCP) --------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// The spin is a C++ loop around a branch-free try_wait so that the compiler knows the lanes of a warp may leave
// it at different times and reconverges them (the warp-collective tcgen05.ld after it needs a converged warp).
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t"
      "}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return ok != 0u;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

}  // namespace chisao
