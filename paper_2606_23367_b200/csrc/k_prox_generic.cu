// k_prox_generic.cu - translation unit of the every-asset prox kernels (any N, lots, caps): the fallback where neither the
// cluster-resident form (prox_res.cuh) nor the streaming form (prox_fast.cuh) applies.
#include "prox.cuh"
#include "kernels.h"

#define PROX_STATIC_SHARED(NW)                                           \
  __shared__ double s_scratch[12 * 32];                                  \
  __shared__ double s_gbin[(NW) * PRISM_MAX_GROUPS];                     \
  __shared__ double s_lamS[PRISM_MAX_GROUPS];                            \
  __shared__ double s_gsum[PRISM_MAX_GROUPS];                            \
  __shared__ int s_selS[2];                                              \
  ProxShared sh = {s_scratch, s_gbin, s_lamS, s_gsum, s_selS, nullptr, nullptr, nullptr};

// generic kernel: any N, lots, per-asset caps.  Persistent: grid <= number of accounts.
template <bool LOTS>
__global__ void __launch_bounds__(512) k_prox(const __grid_constant__ ProxArgs p, int mode) {
  PROX_STATIC_SHARED(16)
  for (int a = blockIdx.x; a < p.A; a += gridDim.x) {
    if (p.ap.done[a]) continue;
    const double gam = p.gamma[a], c = p.ap.c[a];
    const double kappa = p.kappa ? p.kappa[a] : 0.0;
    const double lam_b = kappa + (p.c_buy ? p.c_buy[a] : 0.0);
    SrcGlobal<LOTS> src(p, a, c * gam, p.lo[a], p.hi[a], lam_b);
    prox_body<LOTS>(p, mode, src, a, gam, c, kappa, lam_b, sh, false);
  }
}

// shared-memory-resident kernel: 20 N bytes of dynamic shared memory, no lots, no per-asset caps
__global__ void __launch_bounds__(512, 1) k_prox_smem(const __grid_constant__ ProxArgs p, int mode) {
  extern __shared__ __align__(16) double prox_smem[];
  PROX_STATIC_SHARED(16)
  for (int a = blockIdx.x; a < p.A; a += gridDim.x) {
    if (p.ap.done[a]) continue;
    const double gam = p.gamma[a], c = p.ap.c[a];
    const double kappa = p.kappa ? p.kappa[a] : 0.0;
    const double lam_b = kappa + (p.c_buy ? p.c_buy[a] : 0.0);
    __syncthreads();
    SrcSmem src(p, a, c * gam, p.lo[a], p.hi[a], lam_b, lam_b + kappa, prox_smem);
    prox_body<false>(p, mode, src, a, gam, c, kappa, lam_b, sh, true);
  }
}


#define PROX_SMEM_MAX (208 * 1024)   // dynamic shared memory budget of k_prox_smem (plus ~11 KB static)
size_t prox_generic_smem_max() { return PROX_SMEM_MAX; }
cudaError_t prox_generic_set_attrs() {
  return cudaFuncSetAttribute(k_prox_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PROX_SMEM_MAX);
}
cudaError_t prox_generic_launch(int grid, bool lots, bool smem_form, size_t smem, const ProxArgs& a, int mode, cudaStream_t st) {
  if (lots) k_prox<true><<<grid, 512, 0, st>>>(a, mode);
  else if (!smem_form) k_prox<false><<<grid, 512, 0, st>>>(a, mode);
  else k_prox_smem<<<grid, 512, smem, st>>>(a, mode);
  return cudaGetLastError();
}
