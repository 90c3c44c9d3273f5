// k_prox_stream.cu - translation unit of the streaming form of the prox (prox_fast.cuh: k_prox_stream + k_prox_root),
// used for universes too wide for the cluster-resident form.
#include "prox_fast.cuh"
#include "kernels.h"

#define TRY(e) do { cudaError_t _e = (e); if (_e != cudaSuccess) return _e; } while (0)

size_t prox_stream_smem(int G) { return stream_smem_bytes(G); }
int prox_stream_chunk() { return FAST_CH; }
int prox_stream_warps() { return FAST_NW; }
int prox_stream_idx_bits() { return PROX_META_IDX_BITS; }
size_t prox_stream_entry_bytes() { return sizeof(LiveEnt); }

cudaError_t prox_stream_set_attrs(int G, int nsub) {
  TRY(cudaFuncSetAttribute(k_prox_stream<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem_bytes(G)));
  TRY(cudaFuncSetAttribute(k_prox_stream<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem_bytes(G)));
  TRY(cudaFuncSetAttribute(k_prox_stream<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem_bytes(G)));
  TRY(cudaFuncSetAttribute(k_prox_stream<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem_bytes(G)));
  const size_t smr = root_smem_bytes(G, nsub);
  TRY(cudaFuncSetAttribute(k_prox_root<true, ROOT_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smr));
  TRY(cudaFuncSetAttribute(k_prox_root<false, ROOT_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smr));
  TRY(cudaFuncSetAttribute(k_prox_root<true, ROOT_NT_WIDE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smr));
  TRY(cudaFuncSetAttribute(k_prox_root<false, ROOT_NT_WIDE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smr));
  return cudaSuccess;
}
cudaError_t prox_stream_launch(bool check, int S, int A, int G, const ProxArgs& a, int mode, cudaStream_t st) {
  const dim3 grid((unsigned)S, (unsigned)A);
  const size_t sm = stream_smem_bytes(G), smr = root_smem_bytes(G, 2 * S * FAST_NW);
  if (G == 0) { if (check) k_prox_stream<true, true><<<grid, FAST_NW * 32, sm, st>>>(a); else k_prox_stream<false, true><<<grid, FAST_NW * 32, sm, st>>>(a); }
  else { if (check) k_prox_stream<true, false><<<grid, FAST_NW * 32, sm, st>>>(a); else k_prox_stream<false, false><<<grid, FAST_NW * 32, sm, st>>>(a); }
  TRY(cudaGetLastError());
  // one CTA per account: 128 threads, or 512 when the lists can be long and the accounts are fewer than the SMs (32 / 100 /
  // 148 accounts of configs[2]: 26.7 / 34.2 / 38.8 -> 21.8 / 27.8 / 31.8 ms; see ROOT_WIDE_MAX_A for why not beyond)
  if (a.N >= ROOT_WIDE_MIN_N && A <= ROOT_WIDE_MAX_A) {
    if (check) k_prox_root<true, ROOT_NT_WIDE><<<A, ROOT_NT_WIDE, smr, st>>>(a, mode & ~PROX_CHECK); else k_prox_root<false, ROOT_NT_WIDE><<<A, ROOT_NT_WIDE, smr, st>>>(a, mode);
  } else {
    if (check) k_prox_root<true, ROOT_NT><<<A, ROOT_NT, smr, st>>>(a, mode & ~PROX_CHECK); else k_prox_root<false, ROOT_NT><<<A, ROOT_NT, smr, st>>>(a, mode);
  }
  return cudaGetLastError();
}
cudaError_t prox_rescale_launch(int A, const ProxArgs& a, cudaStream_t st) {
  const unsigned nb = (unsigned)((a.N + RESCALE_PER_CTA - 1) / RESCALE_PER_CTA);
  k_prox_rescale<<<dim3(nb, (unsigned)A), 256, 0, st>>>(a);
  return cudaGetLastError();
}
