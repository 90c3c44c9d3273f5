// k_gemm.cu - translation unit of the factor GEMMs (H1, H3): kernels in gemm.cuh, launch wrappers of kernels.h.
#include "gemm.cuh"
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
  });
  return cudaSuccess;
}

cudaError_t gemm1_launch(int gemm_mode, int mt, int nchunk, int kp, const Gemm1Args& a, cudaStream_t st) {
  if (gemm_mode == 1) {
    dim3 grid(nchunk, (unsigned)(((int64_t)a.A * kp + 127) / 128));
    k_gemm1_ref<<<grid, 128, 0, st>>>(a, kp);
  } else {
    dim3 grid(nchunk, (a.A + G1_TA - 1) / G1_TA);
    MT_SWITCH(mt, k_gemm1<MT><<<grid, 256, g1_smem(MT), st>>>(a));
  }
  return cudaGetLastError();
}

template <int MODE>
static void gemm2_mode(int gemm_mode, int mt, const Gemm2Args& a, cudaStream_t st) {
  if (gemm_mode == 1) {
    dim3 grid((unsigned)((a.N + 127) / 128), a.A);
    k_gemm2_ref<MODE><<<grid, 128, 0, st>>>(a);
  } else {
    dim3 grid((unsigned)((a.N + G2_TN - 1) / G2_TN), (a.A + G2_TM - 1) / G2_TM);
    MT_SWITCH(mt, k_gemm2<MT, MODE><<<grid, 256, g2_smem(MT), st>>>(a));
  }
}
cudaError_t gemm2_launch(int gemm_mode, int mt, int mode, const Gemm2Args& a, cudaStream_t st) {
  if (mode == G2_ADMM) gemm2_mode<G2_ADMM>(gemm_mode, mt, a, st);
  else if (mode == G2_ADMM_CHECK) gemm2_mode<G2_ADMM_CHECK>(gemm_mode, mt, a, st);
  else gemm2_mode<G2_SIGMA>(gemm_mode, mt, a, st);
  return cudaGetLastError();
}
