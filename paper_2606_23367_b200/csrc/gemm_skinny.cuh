// gemm_skinny.cuh - H1 / H3 factor GEMMs for FEW active accounts (nact <= 32): the configs[4] regime (32 accounts x
// 384,800 assets, k = 100) and the tail of every batch after H6 compaction.  With at most two m16 account tiles there is no
// reuse of a universe element across warps, so the shared-memory tiling of gemm_tf32.cuh only adds barriers and a second
// copy of B (hi and lo arrays): here every warp streams ITS rows of the universe straight from global memory into MMA
// fragments, splits them hi / lo in registers (once per element - in the tiled kernels every warp of the CTA would repeat
// it) and never meets a barrier in its main loop.  The universe is read as ONE fp32 array (half the bytes of hi + lo).
// Numerics are those of gemm_tf32.cuh: x_hi = tf32(x), x_lo = tf32(x - x_hi) of the fp32-rounded operand, three MMAs,
// fp32 accumulators, fp64 epilogue.
// Fragment trick: the contraction index of mma.sync.m16n8k8 may be permuted as long as A and B agree.  Lane (g, t) owns
// the four consecutive contraction indices 16 c + 4 t .. + 3 of block c (one 128-bit load per operand row); k-step
// s in {0, 1} of the block uses elements 2 s (as the "t" column) and 2 s + 1 (as the "t + 4" column).
#pragma once
#include "common.cuh"
#include "gemm_args.cuh"
#include "gemm_tf32.cuh"

#define SKINNY_MAX_ACCOUNTS 32     // two m16 tiles

// row stride (floats) of the V hi / lo copies: >= 16 ceil(kp / 16), = 16 mod 32 (128-bit fragment loads of rows g and g + 1
// of a quarter-warp then fall into different halves of the banks)
__host__ __device__ constexpr int sk_ld(int kp) { return ((kp + 15) / 16 * 16) % 32 == 16 ? (kp + 15) / 16 * 16 : (kp + 15) / 16 * 16 + 16; }
// shared memory of GEMM-2: V hi / lo, then the two-stage ring of epilogue operands (v and c pairs, 16 bytes per lane and row)
__host__ __device__ inline size_t sk2_smem(int kp, int mtiles) {
  return (size_t)2 * 16 * mtiles * sk_ld(kp) * sizeof(float) + (size_t)2 * 2 * 2 * mtiles * 128 * 16;
}
__device__ __forceinline__ void sk_cp16(void* smem, const void* gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void sk_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NLEFT>
__device__ __forceinline__ void sk_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NLEFT) : "memory"); }

// GEMM-2 + fused epilogue (G2_ADMM, G2_ADMM_CHECK), contract of k_gemm2_tf32.  128 threads; warp w of the grid walks the
// 8-asset tiles [tile_begin(w), tile_end(w)); the universe rows of the NEXT tile are requested (into registers) before the
// MMAs of the current one, and so are its epilogue operands v, c - by cp.async into a per-lane ring in shared memory,
// because the register file is what bounds the bytes in flight here (each lane copies exactly the 16 bytes it reads later:
// no barrier, only cp.async.wait_group).
template <int NT, int MTILES, int MODE>
__global__ void __launch_bounds__(128) k_gemm2_skinny(Gemm2Args p, const float* __restrict__ Bp32, int tiles_per_warp) {
  extern __shared__ __align__(16) unsigned char sk_raw[];
  constexpr int KP = 8 * NT, K16 = (KP + 15) / 16, LD = sk_ld(KP), ROWS = 16 * MTILES;
  constexpr bool TAIL8 = (KP % 16) != 0;                  // the last block holds 8 indices only
  float* Vh = (float*)sk_raw;                              // [ROWS][LD]
  float* Vl = Vh + (size_t)ROWS * LD;
  double2* ring = (double2*)(Vl + (size_t)ROWS * LD);      // [stage 2][v, c][m][h][128 lanes]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  if (p.nact <= 0) return;
  for (int c = tid; c < ROWS * (LD / 2); c += 128) {       // V = S^-1 T (fp64) -> hi / lo, zero beyond kp
    const int r = c / (LD / 2), cc = (c % (LD / 2)) * 2;
    uint32_t h0 = 0, l0 = 0, h1 = 0, l1 = 0;
    if (cc < KP) {
      const int slot = min(r, p.nact - 1);
      const int a = p.act ? p.act[slot] : slot;
      const double2 v = *(const double2*)(p.V + (int64_t)a * p.ldv + cc);
      tf32_split((float)v.x, h0, l0);
      tf32_split((float)v.y, h1, l1);
    }
    *(uint2*)(Vh + r * LD + cc) = make_uint2(h0, h1);
    *(uint2*)(Vl + r * LD + cc) = make_uint2(l0, l1);
  }
  int arow[MTILES][2], acct[MTILES][2];
  double gsc[MTILES][2], gam[MTILES][2];
#pragma unroll
  for (int m = 0; m < MTILES; ++m)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int slot = 16 * m + g + 8 * h;
      arow[m][h] = slot < p.nact;
      acct[m][h] = arow[m][h] ? (p.act ? p.act[slot] : slot) : 0;
      gam[m][h] = arow[m][h] ? p.gamma[acct[m][h]] : 1.0;
      gsc[m][h] = arow[m][h] ? 1.0 / (gam[m][h] * (1.0 + p.c[acct[m][h]])) : 0.0;
    }
  __syncthreads();
  const int64_t ntile = (p.N + 7) / 8;
  const int64_t wg = (int64_t)blockIdx.x * 4 + warp;
  const int64_t tb = wg * tiles_per_warp, te = min(tb + tiles_per_warp, ntile);
  if (tb >= te) return;
  auto load_B = [&](float4 (&b)[K16], int64_t tile) {
    const float* row = Bp32 + min(tile * 8 + g, p.N - 1) * KP;
#pragma unroll
    for (int c = 0; c < KP / 16; ++c) b[c] = *(const float4*)(row + 16 * c + 4 * t);
    if (TAIL8) {                                           // 8 indices left: lane t owns 2 t, 2 t + 1 - one k-step
      const float2 q = *(const float2*)(row + 16 * (KP / 16) + 2 * t);
      b[K16 - 1] = make_float4(q.x, q.y, 0.f, 0.f);
    }
  };
  auto ring_at = [&](int stage, int arr, int m, int h) { return ring + (size_t)(((stage * 2 + arr) * MTILES + m) * 2 + h) * 128 + tid; };
  auto request_vc = [&](int stage, int64_t tile) {
    const int64_t ib = tile * 8 + 2 * t;
    if (ib >= p.ldw) return;
#pragma unroll
    for (int m = 0; m < MTILES; ++m)
#pragma unroll
      for (int h = 0; h < 2; ++h)
        if (arow[m][h]) {
          const int64_t rowp = (int64_t)acct[m][h] * p.ldw;
          sk_cp16(ring_at(stage, 0, m, h), p.v + rowp + ib);
          sk_cp16(ring_at(stage, 1, m, h), p.cc + rowp + ib);
        }
  };
  float4 bcur[K16], bnext[K16];
  load_B(bcur, tb);
  request_vc(0, tb);
  sk_commit();
  const float* vh = Vh + (size_t)g * LD + 4 * t;
  const float* vl = Vl + (size_t)g * LD + 4 * t;
#pragma unroll 1
  for (int64_t tile = tb; tile < te; ++tile) {
    const int stage = (int)(tile - tb) & 1;
    if (tile + 1 < te) { load_B(bnext, tile + 1); request_vc(stage ^ 1, tile + 1); }
    sk_commit();
    // D[slot 16 m + g (+8)][asset ib, ib + 1]
    const int64_t ib = tile * 8 + 2 * t;
    const bool iin = ib < p.ldw;
    const double2 iv = iin ? *(const double2*)(p.invd + ib) : make_double2(0.0, 0.0);   // (padded with zeros to ldw)
    float acc[MTILES][4];
#pragma unroll
    for (int m = 0; m < MTILES; ++m) { acc[m][0] = acc[m][1] = acc[m][2] = acc[m][3] = 0.f; }
#pragma unroll
    for (int c = 0; c < KP / 16; ++c) {
      uint32_t bh[4], bl[4];
      tf32_split(bcur[c].x, bh[0], bl[0]); tf32_split(bcur[c].y, bh[1], bl[1]);
      tf32_split(bcur[c].z, bh[2], bl[2]); tf32_split(bcur[c].w, bh[3], bl[3]);
#pragma unroll
      for (int m = 0; m < MTILES; ++m) {
        const uint4 h0 = *(const uint4*)(vh + (size_t)(16 * m) * LD + 16 * c), h1 = *(const uint4*)(vh + (size_t)(16 * m + 8) * LD + 16 * c);
        const uint4 l0 = *(const uint4*)(vl + (size_t)(16 * m) * LD + 16 * c), l1 = *(const uint4*)(vl + (size_t)(16 * m + 8) * LD + 16 * c);
        {
          const uint32_t ah[4] = {h0.x, h1.x, h0.y, h1.y}, al[4] = {l0.x, l1.x, l0.y, l1.y};
          mma_tf32(acc[m], al, bh[0], bh[1]);
          mma_tf32(acc[m], ah, bl[0], bl[1]);
          mma_tf32(acc[m], ah, bh[0], bh[1]);
        }
        {
          const uint32_t ah[4] = {h0.z, h1.z, h0.w, h1.w}, al[4] = {l0.z, l1.z, l0.w, l1.w};
          mma_tf32(acc[m], al, bh[2], bh[3]);
          mma_tf32(acc[m], ah, bl[2], bl[3]);
          mma_tf32(acc[m], ah, bh[2], bh[3]);
        }
      }
    }
    if (TAIL8) {
      constexpr int c = K16 - 1;
      uint32_t bh[2], bl[2];
      tf32_split(bcur[c].x, bh[0], bl[0]); tf32_split(bcur[c].y, bh[1], bl[1]);
#pragma unroll
      for (int m = 0; m < MTILES; ++m) {
        const float* th = Vh + (size_t)(16 * m + g) * LD + 16 * c + 2 * t;
        const float* tl = Vl + (size_t)(16 * m + g) * LD + 16 * c + 2 * t;
        const uint2 h0 = *(const uint2*)th, h1 = *(const uint2*)(th + 8 * LD), l0 = *(const uint2*)tl, l1 = *(const uint2*)(tl + 8 * LD);
        const uint32_t ah[4] = {h0.x, h1.x, h0.y, h1.y}, al[4] = {l0.x, l1.x, l0.y, l1.y};
        mma_tf32(acc[m], al, bh[0], bh[1]);
        mma_tf32(acc[m], ah, bl[0], bl[1]);
        mma_tf32(acc[m], ah, bh[0], bh[1]);
      }
    }
    sk_wait<1>();                                           // this tile's v, c have landed (the next tile's group may be in flight)
#pragma unroll
    for (int m = 0; m < MTILES; ++m)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (!arow[m][h] || !iin) continue;
        const int a = acct[m][h];
        const double2 v2 = *ring_at(stage, 0, m, h), c2 = *ring_at(stage, 1, m, h);
        const int64_t rowp = (int64_t)a * p.ldw, i = ib;
        const double b0 = (double)acc[m][2 * h], b1 = (double)acc[m][2 * h + 1];
        const double s0 = b0 * iv.x * gsc[m][h], s1 = b1 * iv.y * gsc[m][h];
        double2 vn;
        vn.x = v2.x + p.relax * (c2.x - s0);
        vn.y = v2.y + p.relax * (c2.y - s1);
        const bool in0 = i < p.N, in1 = i + 1 < p.N;
        if (in1) *(double2*)(p.v + rowp + i) = vn; else if (in0) p.v[rowp + i] = vn.x;
        if (MODE == G2_ADMM_CHECK) {
          const double2 rt2 = *(const double2*)(p.rt + rowp + i);
          const double x0 = rt2.x - s0, x1 = rt2.y - s1;
          if (in0) {
            const double q0 = p.q ? p.q[rowp + i] : -p.mu[(int64_t)a * p.N + i];
            p.xs[rowp + i] = x0;
            p.pxq[rowp + i] = b0 + gam[m][h] * p.d[i] * x0 + q0;
          }
          if (in1) {
            const double q1 = p.q ? p.q[rowp + i + 1] : -p.mu[(int64_t)a * p.N + i + 1];
            p.xs[rowp + i + 1] = x1;
            p.pxq[rowp + i + 1] = b1 + gam[m][h] * p.d[i + 1] * x1 + q1;
          }
        }
      }
#pragma unroll
    for (int c = 0; c < K16; ++c) bcur[c] = bnext[c];
  }
}

// GEMM-1 (contract of k_gemm1_tf32): Tpart[ch][a][j] = sum_{i in chunk ch} Bt[j][i] X[a][i].  grid = nchunk, 128 threads.
// The four warps of a CTA walk the SAME 16-asset blocks of the chunk and own different factor tiles (warp w: tiles w, w + 4,
// ...), so there is no reduction inside the CTA; r~ rows come from global memory (the second to fourth warp hit L1) and
// are rounded to fp32 and split in registers.  The loads of the next block are issued before the MMAs of the current one.
template <int NT, int MTILES>
__global__ void __launch_bounds__(128) k_gemm1_skinny(Gemm1Args p, const float* __restrict__ Bt32) {
  constexpr int NW = (NT + 3) / 4;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  if (warp >= NT || p.nact <= 0) return;
  const int64_t i_begin = (int64_t)blockIdx.x * p.chunk;
  const int64_t i_end = min(i_begin + p.chunk, p.Npad);
  const int nblk = (int)((i_end - i_begin) / 16);
  const double* xrow[MTILES][2];
#pragma unroll
  for (int m = 0; m < MTILES; ++m)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int slot = min(16 * m + g + 8 * h, p.nact - 1);
      const int a = p.act ? p.act[slot] : slot;
      xrow[m][h] = p.X + (int64_t)a * p.ldw + i_begin + 4 * t;
    }
  const float* brow[NW];
#pragma unroll
  for (int j = 0; j < NW; ++j) brow[j] = Bt32 + (int64_t)(8 * min(warp + 4 * j, NT - 1) + g) * p.ldn + i_begin + 4 * t;
  float acc[MTILES][NW][4];
#pragma unroll
  for (int m = 0; m < MTILES; ++m)
#pragma unroll
    for (int j = 0; j < NW; ++j) { acc[m][j][0] = acc[m][j][1] = acc[m][j][2] = acc[m][j][3] = 0.f; }
  auto load_blk = [&](float4 (&b)[NW], double2 (&x)[MTILES][2][2], int blk) {
#pragma unroll
    for (int j = 0; j < NW; ++j) b[j] = *(const float4*)(brow[j] + 16 * blk);
#pragma unroll
    for (int m = 0; m < MTILES; ++m)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        x[m][h][0] = *(const double2*)(xrow[m][h] + 16 * blk);
        x[m][h][1] = *(const double2*)(xrow[m][h] + 16 * blk + 2);
      }
  };
  float4 bcur[NW], bnext[NW];
  double2 xcur[MTILES][2][2], xnext[MTILES][2][2];
  if (nblk > 0) load_blk(bcur, xcur, 0);
#pragma unroll 1
  for (int blk = 0; blk < nblk; ++blk) {
    if (blk + 1 < nblk) load_blk(bnext, xnext, blk + 1);
    uint32_t ah[MTILES][2][4], al[MTILES][2][4];            // [m][k-step][fragment register]
#pragma unroll
    for (int m = 0; m < MTILES; ++m)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        tf32_split((float)xcur[m][h][0].x, ah[m][0][h], al[m][0][h]);
        tf32_split((float)xcur[m][h][0].y, ah[m][0][2 + h], al[m][0][2 + h]);
        tf32_split((float)xcur[m][h][1].x, ah[m][1][h], al[m][1][h]);
        tf32_split((float)xcur[m][h][1].y, ah[m][1][2 + h], al[m][1][2 + h]);
      }
#pragma unroll
    for (int j = 0; j < NW; ++j) {
      if (warp + 4 * j >= NT) continue;
      uint32_t bh[4], bl[4];
      tf32_split(bcur[j].x, bh[0], bl[0]); tf32_split(bcur[j].y, bh[1], bl[1]);
      tf32_split(bcur[j].z, bh[2], bl[2]); tf32_split(bcur[j].w, bh[3], bl[3]);
#pragma unroll
      for (int m = 0; m < MTILES; ++m) {
        mma_tf32(acc[m][j], al[m][0], bh[0], bh[1]);
        mma_tf32(acc[m][j], ah[m][0], bl[0], bl[1]);
        mma_tf32(acc[m][j], ah[m][0], bh[0], bh[1]);
        mma_tf32(acc[m][j], al[m][1], bh[2], bh[3]);
        mma_tf32(acc[m][j], ah[m][1], bl[2], bl[3]);
        mma_tf32(acc[m][j], ah[m][1], bh[2], bh[3]);
      }
    }
#pragma unroll
    for (int j = 0; j < NW; ++j) bcur[j] = bnext[j];
#pragma unroll
    for (int m = 0; m < MTILES; ++m)
#pragma unroll
      for (int h = 0; h < 2; ++h) { xcur[m][h][0] = xnext[m][h][0]; xcur[m][h][1] = xnext[m][h][1]; }
  }
  // D[slot 16 m + g (+8)][factor 8 n + 2 t (+1)]
#pragma unroll
  for (int m = 0; m < MTILES; ++m)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int slot = 16 * m + g + 8 * h;
      if (slot >= p.nact) continue;
      const int a = p.act ? p.act[slot] : slot;
      double* out = p.Tpart + ((int64_t)blockIdx.x * p.A + a) * p.ldv + 2 * t;
#pragma unroll
      for (int j = 0; j < NW; ++j) {
        const int n = warp + 4 * j;
        if (n < NT) *(double2*)(out + n * 8) = make_double2((double)acc[m][j][2 * h], (double)acc[m][j][2 * h + 1]);
      }
    }
}
