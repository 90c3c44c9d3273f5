// gemm.cuh - H1 / H3 factor GEMMs in fp64 on the tensor pipe (mma.sync m8n8k4 f64, "DMMA"),
// with plain-FMA reference kernels of the same contract (settings.gemm_mode = 1) used to validate them.
//
//   GEMM-1 (contraction over assets, split-K):  Tpart[ch][a][j] = sum_{i in chunk ch} Bt[j][i] * X[a][i]
//   GEMM-2 (streaming, K = kp) + fused epilogue: s_i = (B_i . V_a + V_E[a][g_i]) / M_ai ;
//        ADMM:   v <- v + relax (cc - s)          [ = v + relax (x - z) ]
//        +CHECK: xs = rt - s (= x),  pxq = B_i . V_a + gamma_a d_i x_i + q_ai  (= P x + q, since B'x = V_B / (gamma f))
//        SIGMA:  pxq = B_i . V_a + gamma_a d_i X_ai                             (Sigma-apply for the diagnostics, H8)
// Operand layouts (all fp64): Bt factor-major kp x ldn, Bp asset-major N x kp, X / v / cc / rt account-major with
// leading dimension ldw (multiple of 32, zero padded), V account-major with leading dimension ldv.
#pragma once
#include "common.cuh"
#include "gemm_args.cuh"

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int NLEFT>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NLEFT)); }

template <int MT>
__global__ void __launch_bounds__(256) k_gemm1(Gemm1Args p) {
  extern __shared__ __align__(16) double smem[];
  constexpr int KP = 8 * MT;
  double* As = smem;                                   // [STAGES][KP][G1_LD]
  double* Bs = smem + (size_t)G1_STAGES * KP * G1_LD;  // [STAGES][TA][G1_LD]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int a0 = blockIdx.y * G1_TA;                   // first slot of the tile (H6: slots of the active-account list)
  if (a0 >= p.nact) return;
  const int64_t i_begin = (int64_t)blockIdx.x * p.chunk;
  const int64_t i_end = min(i_begin + p.chunk, p.Npad);
  const int nst = (int)((i_end - i_begin) / G1_KS);

  auto load_stage = [&](int st, int64_t i0) {
    double* as = As + (size_t)st * KP * G1_LD;
    double* bs = Bs + (size_t)st * G1_TA * G1_LD;
    for (int c = tid; c < KP * (G1_KS / 2); c += 256) {
      const int r = c / (G1_KS / 2), cc = (c % (G1_KS / 2)) * 2;
      cp_async16(as + r * G1_LD + cc, p.Bt + (int64_t)r * p.ldn + i0 + cc);
    }
    for (int c = tid; c < G1_TA * (G1_KS / 2); c += 256) {
      const int r = c / (G1_KS / 2), cc = (c % (G1_KS / 2)) * 2;
      const int slot = min(a0 + r, p.nact - 1);
      const int a = p.act ? p.act[slot] : slot;
      cp_async16(bs + r * G1_LD + cc, p.X + (int64_t)a * p.ldw + i0 + cc);
    }
  };
  double acc[MT][2];
#pragma unroll
  for (int m = 0; m < MT; ++m) acc[m][0] = acc[m][1] = 0.0;

  for (int s = 0; s < G1_STAGES - 1; ++s) {
    if (s < nst) load_stage(s, i_begin + (int64_t)s * G1_KS);
    cp_async_commit();
  }
  const int fr = lane >> 2, fc = lane & 3;
  for (int s = 0; s < nst; ++s) {
    cp_async_wait<G1_STAGES - 2>();
    __syncthreads();
    const int nx = s + G1_STAGES - 1;
    if (nx < nst) load_stage(nx % G1_STAGES, i_begin + (int64_t)nx * G1_KS);
    cp_async_commit();
    const double* as = As + (size_t)(s % G1_STAGES) * KP * G1_LD;
    const double* bs = Bs + (size_t)(s % G1_STAGES) * G1_TA * G1_LD + (warp * 8 + fr) * G1_LD;
#pragma unroll
    for (int k0 = 0; k0 < G1_KS; k0 += 4) {
      const double b = bs[k0 + fc];
#pragma unroll
      for (int m = 0; m < MT; ++m) dmma884(acc[m][0], acc[m][1], as[(m * 8 + fr) * G1_LD + k0 + fc], b);
    }
  }
  cp_async_wait<0>();
  // D[j = 8m + lane/4][a = a0 + 8 warp + 2 (lane%4) + {0,1}]
#pragma unroll
  for (int m = 0; m < MT; ++m) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int slot = a0 + warp * 8 + fc * 2 + h;
      if (slot < p.nact) {
        const int a = p.act ? p.act[slot] : slot;
        p.Tpart[((int64_t)blockIdx.x * p.A + a) * p.ldv + m * 8 + fr] = acc[m][h];
      }
    }
  }
}

// reference: one thread per (a, j), plain FMA, same chunking.  F32: the precision experiment of DESIGN.md (would a
// TF32x3 / fp32 tensor path hold the tolerance?): both operands rounded to fp32, products and sums in fp32.
template <bool F32>
__global__ void k_gemm1_ref(Gemm1Args p, int kp) {
  const int64_t t = (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
  if (t >= (int64_t)p.nact * kp) return;
  const int slot = (int)(t / kp), j = (int)(t % kp);
  const int a = p.act ? p.act[slot] : slot;
  const int64_t i_begin = (int64_t)blockIdx.x * p.chunk, i_end = min(i_begin + p.chunk, p.Npad);
  double s = 0.0;
  if (F32) {
    float sf = 0.f;
    for (int64_t i = i_begin; i < i_end; ++i) sf = fmaf((float)p.Bt[(int64_t)j * p.ldn + i], (float)p.X[(int64_t)a * p.ldw + i], sf);
    s = (double)sf;
  } else {
    for (int64_t i = i_begin; i < i_end; ++i) s = fma(p.Bt[(int64_t)j * p.ldn + i], p.X[(int64_t)a * p.ldw + i], s);
  }
  p.Tpart[((int64_t)blockIdx.x * p.A + a) * p.ldv + j] = s;
}

// ------------------------------------------------------------------------------------------------ GEMM-2
template <int MODE>
__device__ __forceinline__ void g2_epilogue(const Gemm2Args& p, int a, int64_t i, double bv) {
  const double gam = p.gamma[a];
  const int64_t idx = (int64_t)a * p.ldw + i;
  if (MODE == G2_SIGMA) {
    p.pxq[idx] = bv + gam * p.d[i] * p.X[idx];
    return;
  }
  const double c = p.c[a];
  double uv = bv;
  if (p.G) uv += p.V[(int64_t)a * p.ldv + p.kp + p.group_id[i]];
  const double s = uv * p.invd[i] / (gam * (1.0 + c));
  p.v[idx] = p.v[idx] + p.relax * (p.cc[idx] - s);
  if (MODE == G2_ADMM_CHECK) {
    const double x = p.rt[idx] - s;
    p.xs[idx] = x;
    const double qi = p.q ? p.q[idx] : -p.mu[(int64_t)a * p.N + i];
    p.pxq[idx] = bv + gam * p.d[i] * x + qi;
  }
}

// Tile: 64 accounts x 64 assets per CTA, K = kp.  Warp w owns accounts a0 + 8 w .. + 7 and walks the 64 assets in two
// column groups of 32; the epilogue operands of a group (v, c pairs) are requested BEFORE the group's DMMA loop so
// that their latency overlaps the tensor work, and every access is a 16-byte pair.  61 KB of shared memory and
// <= 85 registers: three CTAs per SM.
template <int MT, int MODE>
__global__ void __launch_bounds__(256, 3) k_gemm2(Gemm2Args p) {
  extern __shared__ __align__(16) double smem[];
  constexpr int KP = 8 * MT, LD = KP + 4;
  double* Vs = smem;                       // [TM][LD]
  double* Bs = smem + (size_t)G2_TM * LD;  // [TN][LD]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int a0 = blockIdx.y * G2_TM;                    // first slot of the tile (H6: slots of the active-account list)
  const int64_t i0 = (int64_t)blockIdx.x * G2_TN;
  if (a0 >= p.nact) return;
  for (int c = tid; c < G2_TM * (KP / 2); c += 256) {
    const int r = c / (KP / 2), cc = (c % (KP / 2)) * 2;
    const int slot = min(a0 + r, p.nact - 1);
    const int a = p.act ? p.act[slot] : slot;
    cp_async16(Vs + r * LD + cc, p.V + (int64_t)a * p.ldv + cc);
  }
  for (int c = tid; c < G2_TN * (KP / 2); c += 256) {
    const int r = c / (KP / 2), cc = (c % (KP / 2)) * 2;
    const int64_t i = min(i0 + r, p.N - 1);
    cp_async16(Bs + r * LD + cc, p.Bp + i * KP + cc);
  }
  cp_async_commit();
  const int fr = lane >> 2, fc = lane & 3;
  const int slot = a0 + warp * 8 + fr;
  const bool arow = slot < p.nact;
  const int a = arow ? (p.act ? p.act[slot] : slot) : 0;
  const bool fastep = MODE != G2_SIGMA && !p.G;          // pair-wise epilogue (the rows are padded to 32: always in range)
  double gsc = 0.0, gam = 0.0;
  if (arow && MODE != G2_SIGMA) { gam = p.gamma[a]; gsc = 1.0 / (gam * (1.0 + p.c[a])); }
  const int64_t rowp = (int64_t)a * p.ldw;
  cp_async_wait<0>();
  __syncthreads();
  const double* vs = Vs + (warp * 8 + fr) * LD;
#pragma unroll 1
  for (int cg = 0; cg < G2_TN / 32; ++cg) {
    // D[a][i = ib + 8 n + 2 fc + {0,1}], n = 0..3
    const int64_t ib = i0 + cg * 32 + fc * 2;
    double2 v2[4], c2[4];
    if (fastep && arow) {
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        if (ib + n * 8 < p.ldw) {
          v2[n] = *(const double2*)(p.v + rowp + ib + n * 8);
          c2[n] = *(const double2*)(p.cc + rowp + ib + n * 8);
        }
      }
    }
    double acc[4][2];
#pragma unroll
    for (int n = 0; n < 4; ++n) acc[n][0] = acc[n][1] = 0.0;
    const double* bs = Bs + (cg * 32 + fr) * LD + fc;
#pragma unroll 2
    for (int k0 = 0; k0 < KP; k0 += 4) {
      const double av = vs[k0 + fc];
#pragma unroll
      for (int n = 0; n < 4; ++n) dmma884(acc[n][0], acc[n][1], av, bs[n * 8 * LD + k0]);
    }
    if (!arow) continue;
    if (fastep) {
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        const int64_t i = ib + n * 8;
        if (i >= p.ldw) continue;
        const double2 iv = *(const double2*)(p.invd + i);                   // (invd is padded with zeros to ldw)
        const double s0 = acc[n][0] * iv.x * gsc, s1 = acc[n][1] * iv.y * gsc;
        double2 vn;
        vn.x = v2[n].x + p.relax * (c2[n].x - s0);
        vn.y = v2[n].y + p.relax * (c2[n].y - s1);
        const bool in0 = i < p.N, in1 = i + 1 < p.N;
        if (in1) *(double2*)(p.v + rowp + i) = vn; else if (in0) p.v[rowp + i] = vn.x;
        if (MODE == G2_ADMM_CHECK) {
          const double2 rt2 = *(const double2*)(p.rt + rowp + i);
          const double x0 = rt2.x - s0, x1 = rt2.y - s1;
          if (in0) {
            const double q0 = p.q ? p.q[rowp + i] : -p.mu[(int64_t)a * p.N + i];
            p.xs[rowp + i] = x0;
            p.pxq[rowp + i] = acc[n][0] + gam * p.d[i] * x0 + q0;
          }
          if (in1) {
            const double q1 = p.q ? p.q[rowp + i + 1] : -p.mu[(int64_t)a * p.N + i + 1];
            p.xs[rowp + i + 1] = x1;
            p.pxq[rowp + i + 1] = acc[n][1] + gam * p.d[i + 1] * x1 + q1;
          }
        }
      }
    } else {
#pragma unroll
      for (int n = 0; n < 4; ++n) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int64_t i = ib + n * 8 + h;
          if (i < p.N) g2_epilogue<MODE>(p, a, i, acc[n][h]);
        }
      }
    }
  }
}

template <int MODE, bool F32>
__global__ void k_gemm2_ref(Gemm2Args p) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N || (int)blockIdx.y >= p.nact) return;
  const int a = p.act ? p.act[blockIdx.y] : (int)blockIdx.y;
  double bv = 0.0;
  if (F32) {
    float bf = 0.f;
    for (int j = 0; j < p.kp; ++j) bf = fmaf((float)p.Bp[i * p.kp + j], (float)p.V[(int64_t)a * p.ldv + j], bf);
    bv = (double)bf;
  } else {
    for (int j = 0; j < p.kp; ++j) bv = fma(p.Bp[i * p.kp + j], p.V[(int64_t)a * p.ldv + j], bv);
  }
  g2_epilogue<MODE>(p, a, i, bv);
}
