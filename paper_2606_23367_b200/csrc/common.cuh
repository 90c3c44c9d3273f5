// common.cuh - problem object, device helpers.  Part of the single translation unit prism.cu.
// Notation follows SURVEY.md 8.0 / 8(a): accounts a, assets i, factors j, groups g; U = [B | E'] and
// x-update (M + U Lambda U') x = r solved through the k' x k' capacitance S = Lambda^-1 + U' M^-1 U.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/prism.h"

#define PRISM_KP_ALIGN 8          // factor dimension padded to the m8n8k4 tile
#define PRISM_MAX_KPRIME 160      // k + G limit of the in-shared-memory capacitance inversion

struct AccountParams {            // per-account scalars, struct of arrays on the device (A entries each)
  double* c;        // rho scale: rho_i = c gamma d_i
  double* alpha;    // buy threshold  nu + theta   (warm start of the root find)
  double* beta;     // sell threshold nu - theta
  int32_t* mode;    // 0: turnover inactive (alpha == beta == nu), 1: cap active
  double* bsum;     // 1 - sum_i w0_i : budget in trade space
  int32_t* done;    // convergence mask (H6)
  int32_t* conv;    // 1 if own tolerance met
  int32_t* iters;
  int32_t* refactor;// 1: capacitance must be rebuilt (rho changed); 2: streaming form - a new rho scale is pending in c_new:
                    // k_prox_rescale rewrites the account's iterate for it, k_factor then adopts it
  double* c_new;    // pending rho scale (refactor == 2)
  int32_t* nadapt;  // iteration of the account's last rho adaptation
  double* win;      // live-list window of the prox for the next launch (threshold units)
  double* wins;     // window of the streaming pass (prox_fast.cuh), >= win
  double* slack;    // band ramp (prox_fast.cuh): largest band violation of the band-free projection at band_start
};

struct prism_problem {
  int64_t N;
  int32_t k, kp, A, G, Kp;       // kp: k padded to 8 * MT; Kp = kp: rows of T and V per account (U = Bp)
  int64_t ldv;                   // leading dimension of V / T rows (Kp padded to 8)
  uint32_t flags;
  int32_t max_lots;
  prism_data d;
  // shared precomputed (owned)
  double* Bp;       // N x kp, asset-major, zero padded            (GEMM-2 operand)
  double* Bt;       // kp x ldn, factor-major                      (GEMM-1 operand)
  float *Bp_hi, *Bp_lo, *Bt_hi, *Bt_lo;   // the universe split for the 3xTF32 GEMMs (gemm_tf32.cuh)
  float *Bp32, *Bt32;                     // the universe rounded to fp32 (N x kp, kp x ldn) for the few-account GEMMs (gemm_skinny.cuh)
  int64_t ldn;      // N padded to 32
  double* invd;     // N
  double* gram;     // Kp x Kp : Bp' D^-1 Bp
  double* q;        // A x N : -mu - gamma Sigma w_b, only with a benchmark shift (else NULL and q = -mu)
  // iterate (owned)
  double *v, *rt, *cc, *xs, *pxq;          // A x N each
  double* Tpart;    // nchunk x A x ldv  split-K partials of GEMM-1
  int32_t nchunk;
  int64_t chunk;    // assets per split-K chunk
  double *V;        // A x ldv
  double *Sinv;     // A x Kp x Kp
  double *gw0, *lamG;     // A x G: group sums of w0; band multipliers
  double *resid;    // A x PRISM_NRES (internal copy)
  double *duals;    // A x PRISM_NDUAL(G)
  int32_t* status;  // A
  double* w_stage;  // A x N staging of the host-buffer lane
  int32_t* i_stage; // A
  AccountParams ap;
  // cluster-resident prox (prox_res.cuh): res != 0 when a slice of the account fits a CTA's shared memory
  int32_t res, res_C, res_SL;
  size_t res_smem;
  // streaming prox (prox_fast.cuh)
  int32_t fast, S, capw;  // fast: the streaming form applies; S slices per account; capacity of one warp's live list
  int64_t slice_len, ldc;
  struct LiveEnt *lraw, *lcomp;
  int32_t *lcnt, *lflag;
  unsigned long long* cbin;
  double* chkp;
  int32_t* act;           // H6 compaction: the accounts not done, ascending (rebuilt after a check that finished accounts)
  int32_t* counters;      // [0] number of done accounts
  int32_t* h_counters;    // pinned host mirror
  int64_t bytes;
  int sm_count;
  double dbar;            // mean of d (host copy at create)
  double prof_ms[PRISM_NKERN];   // per-kernel-class device time of the last profiled solve
  int64_t prof_cnt[PRISM_NKERN];
};

static thread_local char g_err[512] = "";
static int set_err(int code, const char* fmt, const char* a = "", long long b = 0) {
  snprintf(g_err, sizeof(g_err), fmt, a, b);
  return code;
}
#define CUDA_TRY(expr)                                                                          \
  do {                                                                                          \
    cudaError_t _e = (expr);                                                                    \
    if (_e != cudaSuccess) return set_err(PRISM_ERR_CUDA, "CUDA error %s at line %lld", cudaGetErrorString(_e), __LINE__); \
  } while (0)

// ------------------------------------------------------------------------------------------ reductions
__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}
__device__ __forceinline__ double warp_max(double x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x = fmax(x, __shfl_xor_sync(0xffffffffu, x, o));
  return x;
}
__device__ __forceinline__ double warp_min(double x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x = fmin(x, __shfl_xor_sync(0xffffffffu, x, o));
  return x;
}

// Block-wide reduction of NV values per thread with one compile-time operation OP (0 sum, 1 max); the result is
// broadcast to all threads.  `scratch` needs NV * 32 doubles.  Fixed order => deterministic.
template <int OP>
__device__ __forceinline__ double red_op(double a, double b) { return OP == 0 ? a + b : fmax(a, b); }
template <int NV, int OP>
__device__ __forceinline__ void block_reduce(double (&val)[NV], double* scratch) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int q = 0; q < NV; ++q) {
    double x = val[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = red_op<OP>(x, __shfl_xor_sync(0xffffffffu, x, o));
    if (lane == 0) scratch[q * 32 + wid] = x;
  }
  __syncthreads();
  // every warp reduces the per-warp partials itself (no second barrier, no broadcast step)
#pragma unroll
  for (int q = 0; q < NV; ++q) {
    double x = lane < nw ? scratch[q * 32 + lane] : (OP == 0 ? 0.0 : -INFINITY);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = red_op<OP>(x, __shfl_xor_sync(0xffffffffu, x, o));
    val[q] = x;
  }
  __syncthreads();      // scratch may be reused by the next call
}

// Deterministic per-group accumulation (replaces shared-memory atomics, whose order is unspecified):
// lanes holding the same group are summed in ascending lane order, the lowest lane adds the sum to THIS WARP's bin.
// Call from warp-uniform control flow (every lane of the warp, `valid` masks the tail).  bins: [nwarps][ngroups].
__device__ __forceinline__ void warp_group_add(double* bins, int ngroups, int g, double val, bool valid) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int key = valid ? g : (0x40000000 + lane);
  const unsigned m = __match_any_sync(0xffffffffu, key);
  unsigned rem = m;
  double s = 0.0;
  while (__any_sync(0xffffffffu, rem != 0u)) {
    const int src = rem ? (__ffs(rem) - 1) : lane;
    const double x = __shfl_sync(0xffffffffu, val, src);
    if (rem) { s += x; rem &= rem - 1u; }
  }
  if (valid && lane == __ffs(m) - 1) bins[wid * ngroups + g] += s;
  __syncwarp();
}
// sum of the per-warp bins in warp order; call after __syncthreads()
__device__ __forceinline__ double group_total(const double* bins, int ngroups, int g) {
  const int nw = (blockDim.x + 31) >> 5;
  double s = 0.0;
  for (int w = 0; w < nw; ++w) s += bins[w * ngroups + g];
  return s;
}
