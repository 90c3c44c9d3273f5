// kernels.h - host-callable launch wrappers of the kernel families.  Each family lives in its own translation unit
// (k_*.cu) so that the library builds in parallel; prism.cu (C ABI + host driver) calls only these functions.
// Every wrapper returns the cudaError_t of its launch / attribute calls.
#pragma once
#include "common.cuh"
#include "prox.cuh"
#include "diag_args.cuh"
#include "gemm_args.cuh"
#include "small_args.cuh"

// ---- factor GEMMs (k_gemm.cu): fp64 DMMA (gemm_mode 0) or plain FMA (gemm_mode 1)
cudaError_t gemm_set_attrs(int mt);
cudaError_t gemm1_launch(int gemm_mode, int mt, int nchunk, int kp, const Gemm1Args& a, const TfSplit& tf, cudaStream_t st);
cudaError_t gemm2_launch(int gemm_mode, int mt, int mode /* G2_* */, const Gemm2Args& a, const TfSplit& tf, cudaStream_t st);
cudaError_t split_universe_launch(const double* Bp, const double* Bt, int64_t N, int kp, int64_t ldn, float* Bp_hi, float* Bp_lo,
                                  float* Bt_hi, float* Bt_lo, float* Bp32, float* Bt32, cudaStream_t st);

cudaError_t fp64_yardstick(cudaStream_t st, double* sink_dev, int sm_count, double* tflops /* host [2]: DMMA, FMA */);

// ---- small kernels (k_small.cu)
cudaError_t small_set_attrs(int Kp);
cudaError_t setup_shared_launch(const void* B, int is32, const double* d, int64_t N, int k, int kp, int64_t ldn, double* Bp,
                                double* Bt, double* invd, cudaStream_t st);
cudaError_t gram_launch(const double* Bt, int64_t ldn, const double* invd, int64_t N, int kp, double* gram, cudaStream_t st);
cudaError_t init_accounts_launch(const InitArgs& a, cudaStream_t st);
cudaError_t precheck_launch(const PrecheckArgs& a, cudaStream_t st);     // NEXT-4: accounts whose constraint set is empty by inspection
cudaError_t warm_start_launch(const WarmArgs& a, cudaStream_t st);
cudaError_t factor_launch(const double* gram, const double* f, const double* gamma, const AccountParams& ap, int A, int k,
                          int kp, double* Sinv, cudaStream_t st);
cudaError_t solve_launch(const SolveArgs& a, cudaStream_t st);
cudaError_t compact_launch(int A, const int32_t* done, int32_t* act, cudaStream_t st);   // H6: list of the accounts not done
cudaError_t scale_fs_launch(const double* Tpart, int nchunk, int A, int k, int kp, int64_t ldv, const double* f,
                            const double* gamma, double* V, cudaStream_t st);
cudaError_t diff_launch(const double* w, const double* wb, int64_t N, int64_t ldw, int A, double* X, cudaStream_t st);
cudaError_t make_q_launch(const double* mu, const double* gSig, int64_t N, int64_t ldw, int A, double* q, cudaStream_t st);
cudaError_t diag_launch(const DiagArgs& a, bool lots, cudaStream_t st);
cudaError_t status_launch(int A, const double* resid, const int32_t* conv, const int32_t* iters, int timed_out, int late_iter,
                          double gate, int32_t* status, cudaStream_t st);
cudaError_t nan_cols_launch(int A, double* resid, cudaStream_t st);
cudaError_t reduce_partials_launch(const double* Tpart, int nchunk, int A, int k, int64_t ldv, double* T, cudaStream_t st);

// error text of a translation unit other than prism.cu (g_err is per unit): sets prism_last_error(), returns code
int prism_internal_set_error(int code, const char* what, const char* detail);

// ---- cluster-resident prox (k_prox_res_plain.cu, k_prox_res_lots.cu)
bool prox_res_geometry(int64_t N, int G, int* C, int* SL, size_t* smem);
cudaError_t prox_res_set_attrs(bool lots, int C, size_t smem);
cudaError_t prox_res_launch(bool lots, bool check, int C, int A, size_t smem, const ProxArgs& a, int mode, cudaStream_t st);

// ---- streaming prox for universes too wide to be resident (k_prox_stream.cu)
size_t prox_stream_smem(int G);
cudaError_t prox_stream_set_attrs(int G, int nsub);
cudaError_t prox_stream_launch(bool check, int S, int A, int G, const ProxArgs& a, int mode, cudaStream_t st);
cudaError_t prox_rescale_launch(int A, const ProxArgs& a, cudaStream_t st);
int prox_stream_chunk();          // FAST_CH
int prox_stream_warps();          // FAST_NW
int prox_stream_idx_bits();       // PROX_META_IDX_BITS
size_t prox_stream_entry_bytes(); // sizeof(LiveEnt)

// ---- every-asset prox (k_prox_generic.cu): any N, lots, caps; fallback only
cudaError_t prox_generic_set_attrs();
cudaError_t prox_generic_launch(int grid, bool lots, bool smem_form, size_t smem, const ProxArgs& a, int mode, cudaStream_t st);
size_t prox_generic_smem_max();
