// k_noalloc.cu - ONE entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph
// capture, tight serving loops, harnesses that forbid it): prism_factor_exposures_noalloc.
//
// It is a variant of the split-K contraction over assets of H1 (gemm.cuh: k_gemm1 / k_gemm1_ref):
//     T[a][j] = sum_i B[i][j] X[a][i]          (factor exposures B'w of A weight vectors)
// The existing path keeps its split-K partials in workspace that prism_problem_create cudaMallocs (Tpart).  Here the
// partials live in a file-scope static __device__ array of a fixed, modest size: PRISM_NOALLOC_SCRATCH_DOUBLES doubles
// = 4 MiB, which every GPU that loads libprism.so holds until the process exits.
//
// Rules this file follows:
//  - In HOST code the name g_noalloc_scratch is a host-side stand-in, not a device address: a kernel handed it would
//    fault (or silently use the wrong memory where the GPU can reach host memory).  The device address is fetched with
//    cudaGetSymbolAddress, once per device, with that device current, return code checked, and that pointer is what
//    the kernels get.  (Device code below could also name the array directly.)
//  - No cudaMalloc, cudaFree or allocating library routine anywhere in this file; sizes beyond the maximum are
//    rejected with PRISM_ERR_INVALID_ARG and a message that states the limit.
//  - All calls share the array and it keeps the last call's contents.  Every partial a call's reduction reads is
//    written by that same call first (nothing needs to start at zero; stale entries beyond nchunk x A x k are never
//    read).  Two calls that OVERLAP on the GPU (different streams, or graphs replayed concurrently) RACE on it:
//    serialise them (one stream, or an event between them).
#include <mutex>

#include "common.cuh"
#include "kernels.h"

static __device__ __align__(256) double g_noalloc_scratch[PRISM_NOALLOC_SCRATCH_DOUBLES];

#define NOALLOC_MAX_DEVICES 64
static double* g_scratch_dev[NOALLOC_MAX_DEVICES];      // device address of the array, per device ordinal
static bool g_scratch_ok[NOALLOC_MAX_DEVICES];
static std::mutex g_scratch_mutex;

// device address of the scratch array on the CURRENT device (set-up step: once per device)
static int noalloc_scratch(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return prism_internal_set_error(PRISM_ERR_CUDA, "cudaGetDevice failed", cudaGetErrorString(e));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return prism_internal_set_error(PRISM_ERR_INVALID_ARG, "device ordinal beyond the no-alloc table (64)", "");
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_ok[dev]) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
    if (e != cudaSuccess || !ptr) {
      cudaGetLastError();
      return prism_internal_set_error(PRISM_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch) failed", cudaGetErrorString(e));
    }
    g_scratch_dev[dev] = ptr;
    g_scratch_ok[dev] = true;
  }
  *out = g_scratch_dev[dev];
  return PRISM_OK;
}

// partial[ch][a][j] = sum over the assets of chunk ch of B[i][j] X[a][i]; one thread per (a, j), plain FMA in asset order
template <typename TB>
__global__ void __launch_bounds__(128) k_exposure_partial(const TB* __restrict__ B, const double* __restrict__ X, int64_t N, int k,
                                                           int A, int64_t chunk, double* __restrict__ partial) {
  const int64_t t = (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
  if (t >= (int64_t)A * k) return;
  const int a = (int)(t / k), j = (int)(t % k);
  const int64_t i0 = (int64_t)blockIdx.x * chunk, i1 = min(i0 + chunk, N);
  double s = 0.0;
  for (int64_t i = i0; i < i1; ++i) s = fma((double)B[i * k + j], X[(int64_t)a * N + i], s);
  partial[((int64_t)blockIdx.x * A + a) * k + j] = s;
}
// T[a][j] = sum of the partials in chunk order (fixed order: deterministic)
__global__ void __launch_bounds__(128) k_exposure_reduce(const double* __restrict__ partial, int nchunk, int A, int k,
                                                          double* __restrict__ T) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (int64_t)A * k) return;
  double s = 0.0;
  for (int ch = 0; ch < nchunk; ++ch) s += partial[(int64_t)ch * A * k + t];
  T[t] = s;
}

extern "C" int prism_noalloc_init(void) {
  double* ptr = nullptr;
  return noalloc_scratch(&ptr);
}

extern "C" int prism_factor_exposures_noalloc(const void* B, int32_t B_is_fp32, const double* X, int64_t N, int32_t k,
                                              int32_t accounts, void* cuda_stream, double* T_out) {
  if (!B || !X || !T_out) return prism_internal_set_error(PRISM_ERR_INVALID_ARG, "B, X and T_out are mandatory", "");
  if (N < 1 || k < 1 || accounts < 1) return prism_internal_set_error(PRISM_ERR_INVALID_ARG, "N, k, accounts must be >= 1", "");
  const int64_t Ak = (int64_t)accounts * k;
  if (Ak > (int64_t)PRISM_NOALLOC_SCRATCH_DOUBLES)
    return prism_internal_set_error(PRISM_ERR_INVALID_ARG,
                                    "accounts x k exceeds the static scratch of prism_factor_exposures_noalloc "
                                    "(PRISM_NOALLOC_SCRATCH_DOUBLES = 524288 doubles = 4 MiB): split the batch", "");
  double* scratch = nullptr;
  const int r = noalloc_scratch(&scratch);
  if (r != PRISM_OK) return r;
  // split-K: as many chunks as the scratch holds, at most 296 (two per SM), at least 256 assets each
  int64_t nchunk = (int64_t)PRISM_NOALLOC_SCRATCH_DOUBLES / Ak;
  if (nchunk > 296) nchunk = 296;
  const int64_t by_len = (N + 255) / 256;
  if (nchunk > by_len) nchunk = by_len;
  if (nchunk < 1) nchunk = 1;
  const int64_t chunk = (N + nchunk - 1) / nchunk;
  nchunk = (N + chunk - 1) / chunk;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const dim3 grid((unsigned)nchunk, (unsigned)((Ak + 127) / 128));
  if (B_is_fp32) k_exposure_partial<float><<<grid, 128, 0, st>>>((const float*)B, X, N, k, accounts, chunk, scratch);
  else k_exposure_partial<double><<<grid, 128, 0, st>>>((const double*)B, X, N, k, accounts, chunk, scratch);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) {
    k_exposure_reduce<<<(unsigned)((Ak + 127) / 128), 128, 0, st>>>(scratch, (int)nchunk, accounts, k, T_out);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) return prism_internal_set_error(PRISM_ERR_CUDA, "kernel launch failed", cudaGetErrorString(e));
  return PRISM_OK;          // asynchronous on cuda_stream: no synchronisation, no allocation
}
