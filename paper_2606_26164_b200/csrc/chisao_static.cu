// chisao_static.cu -- chisao_stick_test_static (include/chisao.h): Phase 2 of a cycle (Eq. 3) on the
// caller's arrays for callers that may not allocate device memory (code under CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc).  The stick test needs scratch -- ||grad f||_inf per sample and the running f_max -- which the
// context path (launch_stick, chisao_select.cu) keeps in the workspace the caller allocated for chisao_init.  Here the scratch
// is a file-scope device array of fixed size: every GPU that loads the library holds
// CHISAO_STATIC_SCRATCH_BYTES of it until the process exits.  The entry point calls no cudaMalloc / cudaFree and no
// allocating library routine; the array's device address is looked up ONCE per device (cudaGetSymbolAddress with that
// device current) -- in host code the array's name is only a stand-in for the symbol, not an address a kernel could use.
//
// Every call on a device shares the one array and finds the previous call's contents in it: the head (f_max, count) is
// cleared on the stream before the kernels, the per-sample part is overwritten for 0 .. N-1 before it is read.  Two calls that
// overlap on the GPU (different streams, no dependency) therefore RACE; calls on one stream are ordered and safe.
//
// The arithmetic is that of k_ginf_fmax + stick_test (chisao_select.cu), restated on plain pointers: the two paths share
// no state, and tests/test_zz_no_alloc.py checks that they give the same flags.
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include <string>
#include "chisao_device.cuh"

namespace chisao { void set_global_error(const char *msg); }   // chisao_api.cu: what chisao_last_error(NULL) returns

namespace {

constexpr int HEAD_WORDS = 64;                                   // 256 bytes: word 0 f_max (ordered encoding), word 1 n_stuck
constexpr size_t SCRATCH_WORDS = HEAD_WORDS + (size_t)CHISAO_STATIC_MAX_N;
static_assert(SCRATCH_WORDS * 4 == CHISAO_STATIC_SCRATCH_BYTES, "include/chisao.h states the size of the static scratch");

static __device__ __align__(256) uint32_t g_stick_scratch[SCRATCH_WORDS];

constexpr int MAX_DEVICES = 64;
uint32_t *g_scratch_addr[MAX_DEVICES] = {nullptr};   // device address of g_stick_scratch on device k (host-side cache)
std::mutex g_scratch_mutex;

int fail(int code, const std::string &msg) { chisao::set_global_error(msg.c_str()); return code; }

// device address of the scratch array on the CURRENT device; looked up at the first call on that device
int scratch_for_current_device(uint32_t **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(CHISAO_E_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(CHISAO_E_INVALID, "chisao_stick_test_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    uint32_t *p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_stick_scratch);
    if (e != cudaSuccess || !p)
      return fail(CHISAO_E_CUDA, std::string("cudaGetSymbolAddress(g_stick_scratch): ") + cudaGetErrorString(e));
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return CHISAO_OK;
}

// ||grad f(x_i)||_inf per sample (one warp per sample) and f_max over the finite values (Alg. 1, R-13)
__global__ void __launch_bounds__(256) k_static_ginf_fmax(const float *__restrict__ g, const float *__restrict__ f, int N, int d,
                                                          uint32_t *scratch) {
  __shared__ float sh_max[8];
  float *ginf = reinterpret_cast<float *>(scratch + HEAD_WORDS);
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int i = blockIdx.x * 8 + wib;
  float fm = -INFINITY;
  if (i < N) {
    const float *gr = g + (size_t)i * d;
    float gi = 0.0f;
    bool nan = false;
    for (int j = lane; j < d; j += 32) { const float a = fabsf(gr[j]); nan |= !(a == a); gi = fmaxf(gi, a); }
    gi = chisao::warp_max(gi);
    nan = __any_sync(0xffffffffu, nan);
    if (lane == 0) {
      ginf[i] = nan ? NAN : gi;          // a NaN gradient can never pass "< eps_grad"
      const float fi = f[i];
      if (fabsf(fi) <= 3.0e38f) fm = fi;
    }
  }
  if (lane == 0) sh_max[wib] = fm;
  __syncthreads();
  if (threadIdx.x == 0) {
    float mx = sh_max[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) mx = fmaxf(mx, sh_max[w]);
    if (mx > -INFINITY) atomicMax(&scratch[0], chisao::enc_ordered(mx));
  }
}

// stuck_i = (||grad f(x_i)||_inf < eps_grad) and (f(x_i) >= f_max + log delta)   (Eq. 3)
__global__ void __launch_bounds__(256) k_static_stick_flags(const float *__restrict__ f, int N, float eps_grad, float log_delta,
                                                            uint32_t *scratch, uint8_t *stuck, int32_t *n_stuck_out, float *f_max_out) {
  const float *ginf = reinterpret_cast<const float *>(scratch + HEAD_WORDS);
  const float fmax = chisao::dec_ordered(scratch[0]);
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  bool st = false;
  if (i < N) {
    const float fi = f[i];
    st = (ginf[i] < eps_grad) && (fabsf(fi) <= 3.0e38f) && (fi >= fmax + log_delta);
    stuck[i] = st ? 1 : 0;
  }
  const unsigned mk = __ballot_sync(0xffffffffu, st);
  if ((threadIdx.x & 31) == 0 && mk && n_stuck_out) atomicAdd(n_stuck_out, __popc(mk));
  if (i == 0 && f_max_out) *f_max_out = fmax;
}

}  // namespace

extern "C" int chisao_stick_test_static(const float *g_dev, const float *f_dev, int32_t N, int32_t d, float eps_grad,
                                        float log_delta, uint8_t *stuck_dev, int32_t *n_stuck_dev, float *f_max_dev,
                                        void *stream_v) {
  if (N < 0 || d < 1 || d > CHISAO_MAX_D) return fail(CHISAO_E_INVALID, "chisao_stick_test_static: need N >= 0 and d in 1..64");
  if (N > CHISAO_STATIC_MAX_N)
    return fail(CHISAO_E_INVALID, "chisao_stick_test_static: N = " + std::to_string(N) + " exceeds CHISAO_STATIC_MAX_N = " +
                                      std::to_string(CHISAO_STATIC_MAX_N) + " (the static scratch holds one float per sample); "
                                      "use a chisao_ctx with a caller-allocated workspace for larger populations");
  if (N > 0 && (!g_dev || !f_dev || !stuck_dev)) return fail(CHISAO_E_INVALID, "chisao_stick_test_static: null device pointer");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream_v);
  uint32_t *scratch = nullptr;
  const int rc = scratch_for_current_device(&scratch);
  if (rc != CHISAO_OK) return rc;
  // what must start at zero: the f_max word and (if asked for) the caller's counter
  cudaError_t e = cudaMemsetAsync(scratch, 0, HEAD_WORDS * sizeof(uint32_t), st);
  if (e == cudaSuccess && n_stuck_dev) e = cudaMemsetAsync(n_stuck_dev, 0, sizeof(int32_t), st);
  if (e != cudaSuccess) return fail(CHISAO_E_CUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(e));
  if (N > 0) k_static_ginf_fmax<<<(N + 7) / 8, 256, 0, st>>>(g_dev, f_dev, N, d, scratch);
  // (N = 0: one block writes f_max = -inf and leaves the counter at zero)
  k_static_stick_flags<<<N > 0 ? (N + 255) / 256 : 1, 256, 0, st>>>(f_dev, N, eps_grad, log_delta, scratch, stuck_dev, n_stuck_dev,
                                                                  f_max_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(CHISAO_E_CUDA, std::string("chisao_stick_test_static launch: ") + cudaGetErrorString(e));
  return CHISAO_OK;
}
