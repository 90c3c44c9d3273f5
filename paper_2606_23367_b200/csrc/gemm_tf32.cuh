// gemm_tf32.cuh - H1 / H3 factor GEMMs on the TF32 tensor path with the 3xTF32 split (fp32-level accuracy):
//     a b  ~=  a_hi b_hi + a_lo b_hi + a_hi b_lo,   x_hi = tf32(x), x_lo = tf32(x - x_hi),   fp32 accumulators,
// same contracts and the same fp64 epilogue as the DMMA kernels of gemm.cuh.  BASELINE.json:north_star: "TF32 or fp64
// DMMA is chosen against the tolerance"; the choice is measured (with operands and sums in fp32 the
// iteration counts, the weights and the certificates of the parity cases do not move), and with it both GEMMs stop
// being bound by the fp64 pipe: GEMM-1 reads r~ once, GEMM-2 reads v, c and writes v - they are HBM-bound
// (18 flop/B against a ridge of 5.7 flop/B for fp64 and > 100 flop/B for TF32).
// The shared universe B is split once at create (Bt_hi/lo factor-major, Bp_hi/lo asset-major, fp32 storage); the
// per-account operands (r~, V = S^-1 T) are fp64 in memory and are split in registers / on the way to shared memory.
// mma.sync.m16n8k8 (accounts on M): A = the per-account operand (row-major, K contiguous), B = the universe (column-major).
#pragma once
#include "common.cuh"
#include "gemm.cuh"
#include "gemm_args.cuh"

#define T1_KS 32                 // assets per pipeline stage of GEMM-1
#define T1_LDB (T1_KS + 4)       // floats  (conflict-free B-fragment loads: 36 = 4 mod 32)
#define T1_LDX (T1_KS + 4)       // doubles (conflict-free 64-bit A-fragment loads)
#define T1_TA 64                 // accounts per CTA: 4 warps x m16
#define T1_STAGES 3

__device__ __forceinline__ uint32_t tf32_of(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void tf32_split(float x, uint32_t& hi, uint32_t& lo) {
  hi = tf32_of(x);
  lo = tf32_of(x - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

struct TfUniverse {              // the universe split for the TF32 path (fp32 storage, tf32-rounded values)
  const float *Bt_hi, *Bt_lo;    // kp x ldn, factor-major
  const float *Bp_hi, *Bp_lo;    // N x kp, asset-major
};

__host__ __device__ inline size_t t1_smem(int kp) {
  return (size_t)T1_STAGES * ((size_t)2 * kp * T1_LDB * sizeof(float) + (size_t)T1_TA * T1_LDX * sizeof(double));
}

// GEMM-1: Tpart[ch][a][j] = sum_{i in chunk ch} Bt[j][i] X[a][i].  grid = (nchunk, ceil(nact / 64)), 128 threads.
template <int NT>                // NT = kp / 8 factor tiles (n8)
__global__ void __launch_bounds__(128) k_gemm1_tf32(Gemm1Args p, TfUniverse u) {
  extern __shared__ __align__(16) unsigned char t1_raw[];
  constexpr int KP = 8 * NT;
  constexpr size_t STAGE = (size_t)2 * KP * T1_LDB * sizeof(float) + (size_t)T1_TA * T1_LDX * sizeof(double);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const int a0 = blockIdx.y * T1_TA;
  if (a0 >= p.nact) return;
  const int64_t i_begin = (int64_t)blockIdx.x * p.chunk;
  const int64_t i_end = min(i_begin + p.chunk, p.Npad);
  const int nst = (int)((i_end - i_begin) / T1_KS);

  auto load_stage = [&](int st, int64_t i0) {
    unsigned char* sb = t1_raw + (size_t)st * STAGE;
    double* xs = (double*)sb;                                         // [T1_TA][T1_LDX]
    float* bh = (float*)(sb + (size_t)T1_TA * T1_LDX * sizeof(double));   // [KP][T1_LDB]
    float* bl = bh + (size_t)KP * T1_LDB;
    for (int c = tid; c < T1_TA * (T1_KS / 2); c += 128) {
      const int r = c / (T1_KS / 2), cc = (c % (T1_KS / 2)) * 2;
      const int slot = min(a0 + r, p.nact - 1);
      const int a = p.act ? p.act[slot] : slot;
      cp_async16(xs + r * T1_LDX + cc, p.X + (int64_t)a * p.ldw + i0 + cc);
    }
    for (int c = tid; c < KP * (T1_KS / 4); c += 128) {
      const int r = c / (T1_KS / 4), cc = (c % (T1_KS / 4)) * 4;
      cp_async16(bh + r * T1_LDB + cc, u.Bt_hi + (int64_t)r * p.ldn + i0 + cc);
      cp_async16(bl + r * T1_LDB + cc, u.Bt_lo + (int64_t)r * p.ldn + i0 + cc);
    }
  };
  float acc[NT][4];
#pragma unroll
  for (int n = 0; n < NT; ++n) { acc[n][0] = acc[n][1] = acc[n][2] = acc[n][3] = 0.f; }

  for (int s = 0; s < T1_STAGES - 1; ++s) {
    if (s < nst) load_stage(s, i_begin + (int64_t)s * T1_KS);
    cp_async_commit();
  }
  for (int s = 0; s < nst; ++s) {
    cp_async_wait<T1_STAGES - 2>();
    __syncthreads();
    const int nx = s + T1_STAGES - 1;
    if (nx < nst) load_stage(nx % T1_STAGES, i_begin + (int64_t)nx * T1_KS);
    cp_async_commit();
    const unsigned char* sb = t1_raw + (size_t)(s % T1_STAGES) * STAGE;
    const double* xs = (const double*)sb + (size_t)(warp * 16 + g) * T1_LDX + t;
    const float* bh = (const float*)(sb + (size_t)T1_TA * T1_LDX * sizeof(double)) + (size_t)g * T1_LDB + t;
    const float* bl = bh + (size_t)KP * T1_LDB;
#pragma unroll
    for (int k0 = 0; k0 < T1_KS; k0 += 8) {
      uint32_t ah[4], al[4];
      tf32_split((float)xs[k0], ah[0], al[0]);
      tf32_split((float)xs[8 * T1_LDX + k0], ah[1], al[1]);
      tf32_split((float)xs[k0 + 4], ah[2], al[2]);
      tf32_split((float)xs[8 * T1_LDX + k0 + 4], ah[3], al[3]);
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        const uint32_t bh0 = __float_as_uint(bh[n * 8 * T1_LDB + k0]), bh1 = __float_as_uint(bh[n * 8 * T1_LDB + k0 + 4]);
        const uint32_t bl0 = __float_as_uint(bl[n * 8 * T1_LDB + k0]), bl1 = __float_as_uint(bl[n * 8 * T1_LDB + k0 + 4]);
        mma_tf32(acc[n], al, bh0, bh1);
        mma_tf32(acc[n], ah, bl0, bl1);
        mma_tf32(acc[n], ah, bh0, bh1);
      }
    }
  }
  cp_async_wait<0>();
  // D[account = a0 + 16 warp + g (+8)][factor = 8 n + 2 t (+1)]
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int slot = a0 + warp * 16 + g + 8 * h;
    if (slot >= p.nact) continue;
    const int a = p.act ? p.act[slot] : slot;
    double* out = p.Tpart + ((int64_t)blockIdx.x * p.A + a) * p.ldv + 2 * t;
#pragma unroll
    for (int n = 0; n < NT; ++n) *(double2*)(out + n * 8) = make_double2((double)acc[n][2 * h], (double)acc[n][2 * h + 1]);
  }
}

// GEMM-2 + fused epilogue (modes G2_ADMM, G2_ADMM_CHECK; the Sigma-apply of the diagnostics stays on the fp64 kernels).
// A CTA owns 64 accounts and walks `tpc` consecutive 64-asset tiles: V = S^-1 T of its accounts is split ONCE into shared
// memory, the universe tiles are double-buffered with cp.async (the next tile loads during the MMA loop and the
// epilogue of the current one), and the epilogue operands (v, c pairs) are requested before the tile's MMA loop.
// 8 warps: warp w owns accounts 16 (w & 3) .. + 15 and the assets 32 (w >> 2) .. + 31 of the tile.
#define T2_TM 64
#define T2_TN 64
__host__ __device__ inline size_t t2_smem(int kp) { return (size_t)(2 * T2_TM + 4 * T2_TN) * (kp + 4) * sizeof(float); }

template <int NT, int MODE>
__global__ void __launch_bounds__(256, 2) k_gemm2_tf32(Gemm2Args p, TfUniverse u, int tpc) {
  extern __shared__ __align__(16) unsigned char t2_raw[];
  constexpr int KP = 8 * NT, LD = KP + 4;
  float* Vh = (float*)t2_raw;                 // [T2_TM][LD]
  float* Vl = Vh + (size_t)T2_TM * LD;
  float* Bbuf = Vl + (size_t)T2_TM * LD;      // 2 x { hi [T2_TN][LD], lo [T2_TN][LD] }
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const int wr = warp & 3, wc = warp >> 2;
  const int a0 = blockIdx.y * T2_TM;
  if (a0 >= p.nact) return;
  const int64_t ntile = (p.N + T2_TN - 1) / T2_TN;
  const int64_t tile0 = (int64_t)blockIdx.x * tpc;
  const int nt = (int)min((int64_t)tpc, ntile - tile0);
  if (nt <= 0) return;
  auto load_B = [&](int buf, int64_t tile) {
    float* bh = Bbuf + (size_t)buf * 2 * T2_TN * LD;
    float* bl = bh + (size_t)T2_TN * LD;
    const int64_t i0 = tile * T2_TN;
    for (int c = tid; c < T2_TN * (KP / 4); c += 256) {
      const int r = c / (KP / 4), cc = (c % (KP / 4)) * 4;
      const int64_t i = min(i0 + r, p.N - 1);
      cp_async16(bh + r * LD + cc, u.Bp_hi + i * KP + cc);
      cp_async16(bl + r * LD + cc, u.Bp_lo + i * KP + cc);
    }
  };
  load_B(0, tile0);
  cp_async_commit();
  for (int c = tid; c < T2_TM * (KP / 2); c += 256) {      // V is fp64 in memory: split on the way to shared memory
    const int r = c / (KP / 2), cc = (c % (KP / 2)) * 2;
    const int slot = min(a0 + r, p.nact - 1);
    const int a = p.act ? p.act[slot] : slot;
    const double2 v = *(const double2*)(p.V + (int64_t)a * p.ldv + cc);
    uint32_t h0, l0, h1, l1;
    tf32_split((float)v.x, h0, l0);
    tf32_split((float)v.y, h1, l1);
    *(uint2*)(Vh + r * LD + cc) = make_uint2(h0, h1);
    *(uint2*)(Vl + r * LD + cc) = make_uint2(l0, l1);
  }
  int arow[2], acct[2];
  double gsc[2], gam[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int slot = a0 + wr * 16 + g + 8 * h;
    arow[h] = slot < p.nact;
    acct[h] = arow[h] ? (p.act ? p.act[slot] : slot) : 0;
    gam[h] = arow[h] ? p.gamma[acct[h]] : 1.0;
    gsc[h] = arow[h] ? 1.0 / (gam[h] * (1.0 + p.c[acct[h]])) : 0.0;
  }
  const float* vh = Vh + (size_t)(wr * 16 + g) * LD + t;
  const float* vl = Vl + (size_t)(wr * 16 + g) * LD + t;
#pragma unroll 1
  for (int tt = 0; tt < nt; ++tt) {
    cp_async_wait<0>();
    __syncthreads();                                       // tile tt (and, the first time, V) has landed; tile tt - 1 is done with
    if (tt + 1 < nt) load_B((tt + 1) & 1, tile0 + tt + 1);
    cp_async_commit();
    // D[account row g (+8)][asset = ib + 8 n + {0, 1}], n = 0..3
    const int64_t ib = (tile0 + tt) * T2_TN + wc * 32 + 2 * t;
    double2 v2[2][4], c2[2][4], iv4[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) iv4[n] = ib + n * 8 < p.ldw ? *(const double2*)(p.invd + ib + n * 8) : make_double2(0.0, 0.0);   // (padded with zeros to ldw)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int64_t rowp = (int64_t)acct[h] * p.ldw;
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        v2[h][n] = make_double2(0.0, 0.0); c2[h][n] = make_double2(0.0, 0.0);
        if (arow[h] && ib + n * 8 < p.ldw) {
          v2[h][n] = *(const double2*)(p.v + rowp + ib + n * 8);
          c2[h][n] = *(const double2*)(p.cc + rowp + ib + n * 8);
        }
      }
    }
    float acc[4][4];
#pragma unroll
    for (int n = 0; n < 4; ++n) { acc[n][0] = acc[n][1] = acc[n][2] = acc[n][3] = 0.f; }
    const float* bh = Bbuf + (size_t)(tt & 1) * 2 * T2_TN * LD + (size_t)(wc * 32 + g) * LD + t;
    const float* bl = bh + (size_t)T2_TN * LD;
#pragma unroll
    for (int k0 = 0; k0 < KP; k0 += 8) {
      uint32_t ah[4], al[4];
      ah[0] = __float_as_uint(vh[k0]); ah[1] = __float_as_uint(vh[8 * LD + k0]);
      ah[2] = __float_as_uint(vh[k0 + 4]); ah[3] = __float_as_uint(vh[8 * LD + k0 + 4]);
      al[0] = __float_as_uint(vl[k0]); al[1] = __float_as_uint(vl[8 * LD + k0]);
      al[2] = __float_as_uint(vl[k0 + 4]); al[3] = __float_as_uint(vl[8 * LD + k0 + 4]);
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        const uint32_t bh0 = __float_as_uint(bh[n * 8 * LD + k0]), bh1 = __float_as_uint(bh[n * 8 * LD + k0 + 4]);
        const uint32_t bl0 = __float_as_uint(bl[n * 8 * LD + k0]), bl1 = __float_as_uint(bl[n * 8 * LD + k0 + 4]);
        mma_tf32(acc[n], al, bh0, bh1);
        mma_tf32(acc[n], ah, bl0, bl1);
        mma_tf32(acc[n], ah, bh0, bh1);
      }
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      if (!arow[h]) continue;
      const int a = acct[h];
      const int64_t rowp = (int64_t)a * p.ldw;
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        const int64_t i = ib + n * 8;
        if (i >= p.ldw) continue;
        const double b0 = (double)acc[n][2 * h], b1 = (double)acc[n][2 * h + 1];
        const double2 iv = iv4[n];
        const double s0 = b0 * iv.x * gsc[h], s1 = b1 * iv.y * gsc[h];
        double2 vn;
        vn.x = v2[h][n].x + p.relax * (c2[h][n].x - s0);
        vn.y = v2[h][n].y + p.relax * (c2[h][n].y - s1);
        const bool in0 = i < p.N, in1 = i + 1 < p.N;
        if (in1) *(double2*)(p.v + rowp + i) = vn; else if (in0) p.v[rowp + i] = vn.x;
        if (MODE == G2_ADMM_CHECK) {
          const double2 rt2 = *(const double2*)(p.rt + rowp + i);
          const double x0 = rt2.x - s0, x1 = rt2.y - s1;
          if (in0) {
            const double q0 = p.q ? p.q[rowp + i] : -p.mu[(int64_t)a * p.N + i];
            p.xs[rowp + i] = x0;
            p.pxq[rowp + i] = b0 + gam[h] * p.d[i] * x0 + q0;
          }
          if (in1) {
            const double q1 = p.q ? p.q[rowp + i + 1] : -p.mu[(int64_t)a * p.N + i + 1];
            p.xs[rowp + i + 1] = x1;
            p.pxq[rowp + i + 1] = b1 + gam[h] * p.d[i + 1] * x1 + q1;
          }
        }
      }
    }
  }
  cp_async_wait<0>();
}

// universe split at create: Bt_hi/lo (kp x ldn) and Bp_hi/lo (N x kp) from the padded fp64 copies
__global__ void k_split_universe(const double* Bp, const double* Bt, int64_t N, int kp, int64_t ldn, float* Bp_hi, float* Bp_lo,
                                 float* Bt_hi, float* Bt_lo, float* Bp32, float* Bt32) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e < N * kp) {
    uint32_t h, l;
    tf32_split((float)Bp[e], h, l);
    Bp_hi[e] = __uint_as_float(h); Bp_lo[e] = __uint_as_float(l);
    Bp32[e] = (float)Bp[e];
  }
  if (e < (int64_t)kp * ldn) {
    uint32_t h, l;
    tf32_split((float)Bt[e], h, l);
    Bt_hi[e] = __uint_as_float(h); Bt_lo[e] = __uint_as_float(l);
    Bt32[e] = (float)Bt[e];
  }
}
