// k_gemm.cu - translation unit of the factor GEMMs (H1, H3): kernels in gemm.cuh, launch wrappers of kernels.h.
#include "gemm.cuh"
#include "gemm_tf32.cuh"
#include "gemm_skinny.cuh"
#include "kernels.h"

#define MT_SWITCH(mt, ...)                                            \
  switch (mt) {                                                       \
    case 2: { constexpr int MT = 2; __VA_ARGS__; } break;             \
    case 4: { constexpr int MT = 4; __VA_ARGS__; } break;             \
    case 7: { constexpr int MT = 7; __VA_ARGS__; } break;             \
    case 8: { constexpr int MT = 8; __VA_ARGS__; } break;             \
    case 13: { constexpr int MT = 13; __VA_ARGS__; } break;           \
    default: { constexpr int MT = 16; __VA_ARGS__; } break;           \
  }

static size_t g1_smem(int mt) { return (size_t)G1_STAGES * (8 * mt + G1_TA) * G1_LD * sizeof(double); }
static size_t g2_smem(int mt) { return (size_t)(G2_TM + G2_TN) * (8 * mt + 4) * sizeof(double); }
#define TRY(e) do { cudaError_t _e = (e); if (_e != cudaSuccess) return _e; } while (0)

cudaError_t gemm_set_attrs(int mt) {
  MT_SWITCH(mt, {
    TRY(cudaFuncSetAttribute(k_gemm1<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g1_smem(MT)));
    TRY(cudaFuncSetAttribute(k_gemm2<MT, G2_ADMM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g2_smem(MT)));
    TRY(cudaFuncSetAttribute(k_gemm2<MT, G2_ADMM_CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g2_smem(MT)));
    TRY(cudaFuncSetAttribute(k_gemm2<MT, G2_SIGMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g2_smem(MT)));
    TRY(cudaFuncSetAttribute(k_gemm1_tf32<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t1_smem(8 * MT)));
    TRY(cudaFuncSetAttribute(k_gemm2_tf32<MT, G2_ADMM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t2_smem(8 * MT)));
    TRY(cudaFuncSetAttribute(k_gemm2_tf32<MT, G2_ADMM_CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t2_smem(8 * MT)));
    TRY(cudaFuncSetAttribute(k_gemm2_skinny<MT, 1, G2_ADMM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sk2_smem(8 * MT, 1)));
    TRY(cudaFuncSetAttribute(k_gemm2_skinny<MT, 1, G2_ADMM_CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sk2_smem(8 * MT, 1)));
    TRY(cudaFuncSetAttribute(k_gemm2_skinny<MT, 2, G2_ADMM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sk2_smem(8 * MT, 2)));
    TRY(cudaFuncSetAttribute(k_gemm2_skinny<MT, 2, G2_ADMM_CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sk2_smem(8 * MT, 2)));
  });
  return cudaSuccess;
}
cudaError_t split_universe_launch(const double* Bp, const double* Bt, int64_t N, int kp, int64_t ldn, float* Bp_hi, float* Bp_lo,
                                  float* Bt_hi, float* Bt_lo, float* Bp32, float* Bt32, cudaStream_t st) {
  const int64_t n = (int64_t)kp * ldn;          // ldn >= N
  k_split_universe<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(Bp, Bt, N, kp, ldn, Bp_hi, Bp_lo, Bt_hi, Bt_lo, Bp32, Bt32);
  return cudaGetLastError();
}

cudaError_t gemm1_launch(int gemm_mode, int mt, int nchunk, int kp, const Gemm1Args& a, const TfSplit& tf, cudaStream_t st) {
  if (gemm_mode == PRISM_GEMM_TF32X3 && a.nact <= SKINNY_MAX_ACCOUNTS) {
    if (a.nact <= 16) { MT_SWITCH(mt, k_gemm1_skinny<MT, 1><<<nchunk, 128, 0, st>>>(a, tf.Bt32)); }
    else { MT_SWITCH(mt, k_gemm1_skinny<MT, 2><<<nchunk, 128, 0, st>>>(a, tf.Bt32)); }
  } else if (gemm_mode == PRISM_GEMM_TF32X3) {
    TfUniverse u{tf.Bt_hi, tf.Bt_lo, tf.Bp_hi, tf.Bp_lo};
    dim3 grid(nchunk, (a.nact + T1_TA - 1) / T1_TA);
    MT_SWITCH(mt, k_gemm1_tf32<MT><<<grid, 128, t1_smem(8 * MT), st>>>(a, u));
  } else if (gemm_mode >= 1) {
    dim3 grid(nchunk, (unsigned)(((int64_t)a.nact * kp + 127) / 128));
    if (gemm_mode == PRISM_GEMM_FP32_EXPERIMENT) k_gemm1_ref<true><<<grid, 128, 0, st>>>(a, kp); else k_gemm1_ref<false><<<grid, 128, 0, st>>>(a, kp);
  } else {
    dim3 grid(nchunk, (a.nact + G1_TA - 1) / G1_TA);
    MT_SWITCH(mt, k_gemm1<MT><<<grid, 256, g1_smem(MT), st>>>(a));
  }
  return cudaGetLastError();
}

template <int MODE>
static void gemm2_mode(int gemm_mode, int mt, const Gemm2Args& a, const TfSplit& tf, cudaStream_t st) {
  if (gemm_mode == PRISM_GEMM_TF32X3 && MODE != G2_SIGMA && a.nact <= SKINNY_MAX_ACCOUNTS) {
    // few active accounts: every warp streams its own universe rows (gemm_skinny.cuh); about three CTAs per SM, >= 2 tiles per warp
    constexpr int M2 = MODE == G2_SIGMA ? G2_ADMM : MODE;
    const int64_t ntile = (a.N + 7) / 8;
    int64_t tpw = (ntile + (int64_t)12 * tf.sm_count - 1) / ((int64_t)12 * tf.sm_count);
    if (tpw < 2) tpw = 2;
    const unsigned grid = (unsigned)((ntile + 4 * tpw - 1) / (4 * tpw));
    if (a.nact <= 16) { MT_SWITCH(mt, k_gemm2_skinny<MT, 1, M2><<<grid, 128, sk2_smem(8 * MT, 1), st>>>(a, tf.Bp32, (int)tpw)); }
    else { MT_SWITCH(mt, k_gemm2_skinny<MT, 2, M2><<<grid, 128, sk2_smem(8 * MT, 2), st>>>(a, tf.Bp32, (int)tpw)); }
  } else if (gemm_mode == PRISM_GEMM_TF32X3 && MODE != G2_SIGMA) {
    constexpr int M2 = MODE == G2_SIGMA ? G2_ADMM : MODE;
    TfUniverse u{tf.Bt_hi, tf.Bt_lo, tf.Bp_hi, tf.Bp_lo};
    // tiles per CTA: about two waves of CTAs at two CTAs per SM (the split of V is amortised over the CTA's tiles)
    const int64_t ntile = (a.N + T2_TN - 1) / T2_TN, ta = (a.nact + T2_TM - 1) / T2_TM;
    int tpc = (int)((ntile * ta + (int64_t)4 * tf.sm_count - 1) / ((int64_t)4 * tf.sm_count));
    if (tpc < 1) tpc = 1;
    if (tpc > 16) tpc = 16;
    dim3 grid((unsigned)((ntile + tpc - 1) / tpc), (unsigned)ta);
    MT_SWITCH(mt, k_gemm2_tf32<MT, M2><<<grid, 256, t2_smem(8 * MT), st>>>(a, u, tpc));
  } else if (gemm_mode == 1 || gemm_mode == 2) {
    dim3 grid((unsigned)((a.N + 127) / 128), a.nact);
    if (gemm_mode == PRISM_GEMM_FP32_EXPERIMENT) k_gemm2_ref<MODE, true><<<grid, 128, 0, st>>>(a); else k_gemm2_ref<MODE, false><<<grid, 128, 0, st>>>(a);
  } else {
    dim3 grid((unsigned)((a.N + G2_TN - 1) / G2_TN), (a.nact + G2_TM - 1) / G2_TM);
    MT_SWITCH(mt, k_gemm2<MT, MODE><<<grid, 256, g2_smem(MT), st>>>(a));
  }
}
cudaError_t gemm2_launch(int gemm_mode, int mt, int mode, const Gemm2Args& a, const TfSplit& tf, cudaStream_t st) {
  if (mode == G2_ADMM) gemm2_mode<G2_ADMM>(gemm_mode, mt, a, tf, st);
  else if (mode == G2_ADMM_CHECK) gemm2_mode<G2_ADMM_CHECK>(gemm_mode, mt, a, tf, st);
  else gemm2_mode<G2_SIGMA>(gemm_mode, mt, a, tf, st);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ fp64 yardstick
// Register-resident loops with no memory traffic: what the fp64 tensor pipe (mma.sync m8n8k4 DMMA) and the fp64 FMA pipe
// of THIS device sustain.  bench.py quotes the factor GEMMs against these ("measure a yardstick on the box").
__global__ void __launch_bounds__(256) k_yard_dmma(int iters, double* sink) {
  double acc[8][2];
#pragma unroll
  for (int m = 0; m < 8; ++m) { acc[m][0] = 0.0; acc[m][1] = 0.0; }
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int m = 0; m < 8; ++m) dmma884(acc[m][0], acc[m][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int m = 0; m < 8; ++m) s += acc[m][0] + acc[m][1];
  if (s == 123.456) sink[0] = s;          // keeps the loop alive
}
__global__ void __launch_bounds__(256) k_yard_fma(int iters, double* sink) {
  double acc[8];
#pragma unroll
  for (int m = 0; m < 8; ++m) acc[m] = 1e-3 * m;
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int m = 0; m < 8; ++m) acc[m] = fma(acc[m], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int m = 0; m < 8; ++m) s += acc[m];
  if (s == 123.456) sink[0] = s;
}
// tflops[0] = DMMA, tflops[1] = FMA (2 flops per multiply-add); best of 5 launches each, CUDA events on `st`
cudaError_t fp64_yardstick(cudaStream_t st, double* sink_dev, int sm_count, double* tflops) {
  cudaEvent_t e0, e1;
  TRY(cudaEventCreate(&e0)); TRY(cudaEventCreate(&e1));
  const int iters = 4096, grid = sm_count * 8, nt = 256;
  for (int which = 0; which < 2; ++which) {
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
      cudaEventRecord(e0, st);
      if (which == 0) k_yard_dmma<<<grid, nt, 0, st>>>(iters, sink_dev); else k_yard_fma<<<grid, nt, 0, st>>>(iters, sink_dev);
      cudaEventRecord(e1, st);
      TRY(cudaEventSynchronize(e1));
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep > 0 && ms < best) best = ms;
    }
    // DMMA m8n8k4: 8*8*4 multiply-adds per warp instruction; FMA: one per thread
    const double per_thread_block = which == 0 ? 8.0 * (8 * 8 * 4) * 2.0 * (nt / 32) : 8.0 * 2.0 * nt;
    tflops[which] = per_thread_block * (double)iters * (double)grid / (best * 1e-3) / 1e12;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return cudaGetLastError();
}
