// gemm_args.cuh - argument blocks and tile constants of the factor GEMMs (gemm.cuh)
#pragma once
#include <stdint.h>

#define G1_KS 32           // assets per pipeline stage
#define G1_LD (G1_KS + 4)  // smem row stride (doubles): conflict-free 64-bit fragment loads
#define G1_TA 64           // accounts per CTA (8 warps x one m8n8 column tile)
#define G1_STAGES 3

struct Gemm1Args {
  const double* Bt; int64_t ldn;
  const double* X; int64_t ldw;
  double* Tpart; int64_t ldv;
  int32_t A; int64_t chunk; int64_t Npad;
  // H6 compaction: tile rows are SLOTS of the active-account list; act[slot] = account (NULL: identity, nact = A)
  const int32_t* act; int32_t nact;
};


enum { G2_ADMM = 0, G2_ADMM_CHECK = 1, G2_SIGMA = 2 };
#define G2_TM 64     // accounts per CTA
#define G2_TN 64     // assets per CTA

struct Gemm2Args {
  const double* Bp; int32_t kp;
  const double* V; int64_t ldv;
  int64_t N, ldw; int32_t A, G;
  const uint8_t* group_id;
  const double *invd, *d, *gamma, *c;
  double* v; const double* cc; const double* rt;
  double *xs, *pxq;
  const double *q, *mu;       // q (ldw) or mu (ld N)
  const double* X;            // SIGMA: the vector Sigma is applied to (ldw)
  double relax;
  const int32_t* act; int32_t nact;   // as in Gemm1Args
};


// the universe split for the 3xTF32 kernels (gemm_tf32.cuh): tf32-rounded values in fp32 storage, built at create
struct TfSplit {
  const float *Bt_hi, *Bt_lo;   // kp x ldn, factor-major
  const float *Bp_hi, *Bp_lo;   // N x kp, asset-major
  const float *Bp32, *Bt32;     // the unsplit fp32 copies (gemm_skinny.cuh)
  int sm_count;
};
