// k_small.cu - translation unit of the small kernels: setup (H0), cold start, capacitance factorisation (H0/H7),
// small solves (H2), Sigma-apply glue and the external diagnostics / statuses (H8, H9).
#include "small.cuh"
#include "diag.cuh"
#include "kernels.h"

#define TRY(e) do { cudaError_t _e = (e); if (_e != cudaSuccess) return _e; } while (0)

cudaError_t small_set_attrs(int Kp) {
  TRY(cudaFuncSetAttribute(k_factor, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)Kp * Kp * sizeof(double))));
  return cudaSuccess;
}
cudaError_t setup_shared_launch(const void* B, int is32, const double* d, int64_t N, int k, int kp, int64_t ldn, double* Bp,
                                double* Bt, double* invd, cudaStream_t st) {
  k_setup_shared<<<(unsigned)((N + 127) / 128), 128, 0, st>>>(B, is32, d, N, k, kp, ldn, Bp, Bt, invd);
  return cudaGetLastError();
}
cudaError_t gram_launch(const double* Bt, int64_t ldn, const double* invd, int64_t N, int kp, double* gram, cudaStream_t st) {
  k_gram<<<dim3(kp, kp), 256, 0, st>>>(Bt, ldn, nullptr, invd, N, kp, 0, gram);
  return cudaGetLastError();
}
cudaError_t init_accounts_launch(const InitArgs& a, cudaStream_t st) {
  k_init_accounts<<<a.A, 256, 0, st>>>(a);
  return cudaGetLastError();
}
cudaError_t precheck_launch(const PrecheckArgs& a, cudaStream_t st) {
  k_precheck<<<a.A, 256, 0, st>>>(a);
  return cudaGetLastError();
}
cudaError_t warm_start_launch(const WarmArgs& a, cudaStream_t st) {
  k_warm_start<<<dim3((unsigned)((a.N + 255) / 256), a.A), 256, 0, st>>>(a);
  return cudaGetLastError();
}
cudaError_t factor_launch(const double* gram, const double* f, const double* gamma, const AccountParams& ap, int A, int k,
                          int kp, double* Sinv, cudaStream_t st) {
  k_factor<<<A, 256, (size_t)kp * kp * sizeof(double), st>>>(gram, f, gamma, ap, k, kp, 0, Sinv);
  return cudaGetLastError();
}
cudaError_t solve_launch(const SolveArgs& a, cudaStream_t st) {
  if (a.nchunk >= 128 && a.nact * SOLVE_CL <= 148) {       // few accounts, many chunks: a cluster of CTAs per account
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(a.nact * SOLVE_CL), 1, 1);
    cfg.blockDim = dim3(1024, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = SOLVE_CL; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_solve_cluster, a);
  }
  if (a.nchunk > 64 && a.kp > 64) k_solve<1024><<<a.nact, 1024, 0, st>>>(a);
  else k_solve<256><<<a.nact, 256, 0, st>>>(a);
  return cudaGetLastError();
}
// H6 compaction: act[0 .. n) = the accounts that are not done, ascending (one CTA, ballot scan: a fixed order).
__global__ void __launch_bounds__(1024) k_compact(int A, const int32_t* done, int32_t* act) {
  __shared__ int wsum[32];
  __shared__ int base_s;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid == 0) base_s = 0;
  __syncthreads();
  for (int a0 = 0; a0 < A; a0 += 1024) {
    const int a = a0 + tid;
    const bool live = a < A && !done[a];
    const unsigned m = __ballot_sync(0xffffffffu, live);
    if (lane == 0) wsum[wid] = __popc(m);
    __syncthreads();
    int off = base_s;
    for (int w = 0; w < wid; ++w) off += wsum[w];
    if (live) act[off + __popc(m & ((1u << lane) - 1u))] = a;
    __syncthreads();
    if (tid == 0) { int t = 0; for (int w = 0; w < 32; ++w) t += wsum[w]; base_s += t; }
    __syncthreads();
  }
}
cudaError_t compact_launch(int A, const int32_t* done, int32_t* act, cudaStream_t st) {
  k_compact<<<1, 1024, 0, st>>>(A, done, act);
  return cudaGetLastError();
}
cudaError_t scale_fs_launch(const double* Tpart, int nchunk, int A, int k, int kp, int64_t ldv, const double* f,
                            const double* gamma, double* V, cudaStream_t st) {
  k_scale_fs<<<A, 128, 0, st>>>(Tpart, nchunk, A, k, kp, ldv, f, gamma, V);
  return cudaGetLastError();
}
cudaError_t diff_launch(const double* w, const double* wb, int64_t N, int64_t ldw, int A, double* X, cudaStream_t st) {
  k_diff<<<dim3((unsigned)((N + 255) / 256), A), 256, 0, st>>>(w, wb, N, ldw, X);
  return cudaGetLastError();
}
cudaError_t make_q_launch(const double* mu, const double* gSig, int64_t N, int64_t ldw, int A, double* q, cudaStream_t st) {
  k_make_q<<<dim3((unsigned)((N + 255) / 256), A), 256, 0, st>>>(mu, gSig, N, ldw, q);
  return cudaGetLastError();
}
cudaError_t diag_launch(const DiagArgs& a, bool lots, cudaStream_t st) {
  if (lots) k_diag<true><<<a.A, 256, 0, st>>>(a);
  else k_diag<false><<<a.A, 256, 0, st>>>(a);
  return cudaGetLastError();
}
cudaError_t status_launch(int A, const double* resid, const int32_t* conv, const int32_t* iters, int timed_out, int late_iter,
                          double gate, int32_t* status, cudaStream_t st) {
  k_status<<<(A + 127) / 128, 128, 0, st>>>(A, resid, conv, iters, timed_out, late_iter, gate, status);
  return cudaGetLastError();
}
// prism_residuals: the solver-only columns of the residual block are NaN
__global__ void k_nan_cols(int A, double* resid) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= A) return;
  double* r = resid + (int64_t)a * PRISM_NRES;
  r[PRISM_R_PRIMAL] = NAN; r[PRISM_R_DUAL] = NAN; r[PRISM_R_RHO] = NAN; r[PRISM_R_RESERVED] = 0.0;
}
cudaError_t nan_cols_launch(int A, double* resid, cudaStream_t st) {
  k_nan_cols<<<(A + 127) / 128, 128, 0, st>>>(A, resid);
  return cudaGetLastError();
}
// T[a][j] = sum over the split-K chunks of Tpart[ch][a][j] in chunk order, j < k (prism_factor_exposures)
__global__ void k_reduce_partials(const double* Tpart, int nchunk, int A, int k, int64_t ldv, double* T) {
  const int a = blockIdx.x;
  for (int j = threadIdx.x; j < k; j += blockDim.x) {
    double s = 0.0;
    for (int ch = 0; ch < nchunk; ++ch) s += Tpart[((int64_t)ch * A + a) * ldv + j];
    T[(int64_t)a * k + j] = s;
  }
}
cudaError_t reduce_partials_launch(const double* Tpart, int nchunk, int A, int k, int64_t ldv, double* T, cudaStream_t st) {
  k_reduce_partials<<<A, 128, 0, st>>>(Tpart, nchunk, A, k, ldv, T);
  return cudaGetLastError();
}
