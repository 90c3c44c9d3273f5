// k_prox_res.cu - geometry and dispatch of the cluster-resident prox (prox_res.cuh); the four kernel instantiations
// live in k_prox_res_{00,01,10,11}.cu.
#include "kernels.h"
#include "prox_res.cuh"

#define DECL(lc)                                               \
  cudaError_t prox_res_attrs_##lc(int C, size_t smem);         \
  cudaError_t prox_res_launch_##lc(int C, int A, size_t smem, const ProxArgs& a, int mode, cudaStream_t st);
DECL(00) DECL(01) DECL(10) DECL(11)

// smallest cluster size for which a slice of the account fits the shared-memory budget
bool prox_res_geometry(int64_t N, int G, int* C_out, int* SL_out, size_t* smem_out) {
  static const int kC[] = {1, 2, 4, 8, 16};
  for (int C : kC) {
    int SL = 0;
    if (res_fits(N, G, C, &SL)) {
      *C_out = C; *SL_out = SL; *smem_out = res_layout(SL, G, C).bytes;
      return true;
    }
  }
  return false;
}
cudaError_t prox_res_set_attrs(bool lots, int C, size_t smem) {
  cudaError_t e = lots ? prox_res_attrs_10(C, smem) : prox_res_attrs_00(C, smem);
  if (e != cudaSuccess) return e;
  return lots ? prox_res_attrs_11(C, smem) : prox_res_attrs_01(C, smem);
}
cudaError_t prox_res_launch(bool lots, bool check, int C, int A, size_t smem, const ProxArgs& a, int mode, cudaStream_t st) {
  if (lots) return check ? prox_res_launch_11(C, A, smem, a, mode, st) : prox_res_launch_10(C, A, smem, a, mode, st);
  return check ? prox_res_launch_01(C, A, smem, a, mode, st) : prox_res_launch_00(C, A, smem, a, mode, st);
}
