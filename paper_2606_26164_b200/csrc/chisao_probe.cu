// chisao_probe.cu -- pipe-rate probes behind chisao_measure_peak (include/chisao.h): hand-written micro-benchmarks of
// the FP32 FMA pipe and of the special-function unit, run on the caller's stream and timed with CUDA events.  They give
// the denominators of the "alu" rooflines bench.py reports ("to be measured by FFMA / MUFU
// micro-benchmarks in the same run, because clocks under load differ"); nothing of the CHISAO path depends on them.
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/chisao.h"

namespace {

constexpr int PROBE_THREADS = 256;
constexpr int PROBE_CHAINS = 8;        // independent dependency chains per thread (FFMA latency 4: 2 warps x 8 chains cover it)
constexpr int PROBE_INNER = 64;

// 2 flop per FFMA; every chain is a dependent sequence a <- a * b + c (values stay bounded: |b| < 1)
__global__ void __launch_bounds__(PROBE_THREADS) k_probe_ffma(float *out, int outer, float b, float c) {
  float a[PROBE_CHAINS];
#pragma unroll
  for (int k = 0; k < PROBE_CHAINS; ++k) a[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (int o = 0; o < outer; ++o) {
#pragma unroll
    for (int i = 0; i < PROBE_INNER; ++i)
#pragma unroll
      for (int k = 0; k < PROBE_CHAINS; ++k) a[k] = fmaf(a[k], b, c);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < PROBE_CHAINS; ++k) s += a[k];
  if (s == 123.456f) out[0] = s;       // never true: keeps the chains alive
}

// one MUFU.EX2 per step, chained through a cheap FMUL so that the argument stays in (-1, 0)
__global__ void __launch_bounds__(PROBE_THREADS) k_probe_mufu(float *out, int outer) {
  float a[PROBE_CHAINS];
#pragma unroll
  for (int k = 0; k < PROBE_CHAINS; ++k) a[k] = -(float)(threadIdx.x % 7 + k + 1) * 0.01f;
  for (int o = 0; o < outer; ++o) {
#pragma unroll
    for (int i = 0; i < PROBE_INNER; ++i)
#pragma unroll
      for (int k = 0; k < PROBE_CHAINS; ++k) {
        float e;
        asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(a[k]));
        a[k] = e * -0.5f;
      }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < PROBE_CHAINS; ++k) s += a[k];
  if (s == 123.456f) out[0] = s;
}

}  // namespace

extern "C" int chisao_measure_peak(int32_t which, float *scratch_dev, void *stream_v, double *value) {
  if (!value || !scratch_dev || (which != CHISAO_PEAK_FP32_FMA && which != CHISAO_PEAK_SFU)) return CHISAO_E_INVALID;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream_v);
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
    return CHISAO_E_CUDA;
  const int grid = sms * 8, outer = 256;
  cudaEvent_t a, b;
  if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return CHISAO_E_CUDA;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {   // rep 0 warms up; best of the rest
    cudaEventRecord(a, st);
    if (which == CHISAO_PEAK_FP32_FMA) k_probe_ffma<<<grid, PROBE_THREADS, 0, st>>>(scratch_dev, outer, 0.999f, 1e-3f);
    else k_probe_mufu<<<grid, PROBE_THREADS, 0, st>>>(scratch_dev, outer);
    cudaEventRecord(b, st);
    if (cudaEventSynchronize(b) != cudaSuccess) { cudaEventDestroy(a); cudaEventDestroy(b); return CHISAO_E_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    const double ops = (double)grid * PROBE_THREADS * PROBE_CHAINS * PROBE_INNER * (double)outer;
    const double rate = (which == CHISAO_PEAK_FP32_FMA ? 2.0 : 1.0) * ops / ((double)ms * 1e-3) / 1e12;
    if (rep > 0 && rate > best) best = rate;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  *value = best;
  return cudaGetLastError() == cudaSuccess ? CHISAO_OK : CHISAO_E_CUDA;
}
