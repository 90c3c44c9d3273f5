// prox_fast.cuh - the streaming form of the fused proximal / projection step for the
// configurations without tax lots and per-asset caps: two kernels per iteration.
//
//   k_prox_stream  (HBM-bound, grid = slices x accounts)  ONE pass over the account's assets.  Every asset whose buy
//       and sell amounts cannot change while the thresholds (alpha, beta, lambda_g) stay inside the window
//       [warm start +- W] ("dead": on the kink, clamped at a bound, excluded) is finished on the spot: its output
//       (r~ = M^-1 r, c = r~ - z) is written, its residual terms are accumulated, its constant trade is added to
//       per-group fixed-point bins (integer atomics: the sum does not depend on the order => deterministic).
//       The other assets ("live", a few percent at most once the iteration has settled) are appended to per-warp
//       lists in global memory, each list in ascending asset order.  The streamed arrays reach shared memory
//       through a bulk-copy (TMA engine) pipeline with full / empty mbarriers.
//   k_prox_root    (latency-bound, one CTA per account)  compacts the lists in a fixed order, solves the
//       piecewise-linear equations for (alpha, beta, lambda_g) on the live assets only (prox_rootfind), writes the
//       live assets' outputs, finishes the residual check (convergence mask, H6), and commits the account's state.
//       If the solution left the window, rho has to change, or a NaN shows up, the same CTA redoes the account with
//       the generic every-asset source (prox_body over SrcGlobal): no account state has been touched before that.
#pragma once
#include "prox.cuh"

#define PRISM_FIX_SCALE 1152921504606846976.0            // 2^60
#define PRISM_FIX_INV (1.0 / 1152921504606846976.0)
#define PROX_META_IDX_BITS 22                            // meta = idx | gid << 22 | cls << 30

struct __align__(16) LiveEnt { double T, w0, ir; uint32_t meta, pad; };   // one live asset (32 bytes)

#define FAST_NW 8            // warps per streaming CTA
#define FAST_CH 512          // assets per pipeline stage (two per thread)
#define FAST_NST 3           // stages of the bulk-copy pipeline
#define FAST_STAGE_BYTES (5 * FAST_CH * 8 + 2 * FAST_CH)
#define ROOT_NT 128          // threads of a root CTA
#ifndef ROOT_NT_WIDE
#define ROOT_NT_WIDE 512     // ... from 4,096 instruments on when the accounts are fewer than the SMs (one CTA per account: the idle SMs cannot help, width can)
#endif
#define ROOT_MAXW (ROOT_NT_WIDE / 32)   // warps the per-warp arrays of the root kernel are sized for
#ifndef ROOT_WIDE_MIN_N
#define ROOT_WIDE_MIN_N 4096
#endif
#ifndef ROOT_WIDE_MAX_A
#define ROOT_WIDE_MAX_A 148   // fewer accounts than SMs.  Beyond, width still helps ONE batch (200 / 296 / 400 / 500 accounts of configs[2]:
                              // -11% / -9% / -5% / -1%) but one 512-thread CTA per SM leaves no room for a second batch in flight:
                              // four resident batches of 500 at once 134 -> 165 ms, the 2,000-account queue in four lanes 282 -> 381 ms
#endif
#define ROOT_SCAP 512         // a sorted list up to this length is kept in shared memory (no global-load latency per pass)

__host__ __device__ inline size_t stream_smem_bytes(int G) {
  return (size_t)FAST_NST * FAST_STAGE_BYTES + 2 * FAST_NST * 8 + (size_t)(G > 0 ? G : 1) * 8 + 8 * 32 * 8 + 16;
}

// mbarrier + bulk-copy (TMA engine, 1-D) primitives: global -> shared staging of the streamed arrays
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok = 0;
  const uint32_t addr = smem_u32(bar);
  while (!ok) {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
  }
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ------------------------------------------------------------------------------------------------ streaming kernel
// grid = (slices, accounts), block = 256.  Needs N % 16 == 0 (every row of every streamed array 16-byte aligned).
template <bool CHECK, bool SB>    // SB: no groups - per-CTA fixed-point bins in shared memory (see sbin)
__global__ void __launch_bounds__(FAST_NW * 32, 3) k_prox_stream(const __grid_constant__ ProxArgs p) {
  extern __shared__ __align__(16) unsigned char stream_raw[];
  __shared__ double cst[12];
  // fixed-point bins of this CTA (dead bins, then speculative bins), used when the problem has no groups (one bin per side
  // and account): the constant trades are added up in shared memory and reach the account's global bins with ONE atomic
  // per bin and CTA.  (Per-asset global atomics on one address per
  // account serialise in L2: on configs[4], where a quarter of the 384,800 assets is sold out or at its cap, they held
  // the whole kernel at 1.2 TB/s - the bulk copies queued behind them.)  Integer sums: the order does not matter.
  __shared__ unsigned long long sbin[SB ? 4 : 1];
  const int a = blockIdx.y, sl = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int G = p.G, Gb = G > 0 ? G : 1;
  // A CTA lives for a few chunks only, so its start-up must not be a chain of dependent loads: the account's twelve
  // constants are fetched by twelve lanes of warp 1 at the same time as the done flag, the band multipliers by
  // warp 2.., and thread 0 starts the first bulk copies as soon as it has seen the flag.
  double cv = 0.0;
  if (wid == 1 && lane < 12) {
    switch (lane) {
      case 0: cv = p.lo[a]; break;
      case 1: cv = p.hi[a]; break;
      case 2: cv = p.ap.wins[a]; break;
      case 3: cv = p.ap.win[a]; break;
      case 4: cv = p.gamma[a]; break;
      case 5: cv = p.ap.c[a]; break;
      case 6: cv = p.kappa ? p.kappa[a] : 0.0; break;
      case 7: cv = p.c_buy ? p.c_buy[a] : 0.0; break;
      case 8: cv = p.tau ? p.tau[a] : INFINITY; break;
      case 9: cv = p.ap.alpha[a]; break;
      case 10: cv = p.ap.beta[a]; break;
      default: cv = (double)p.ap.mode[a]; break;
    }
  }
  double lam_mine = 0.0;
  if (tid >= 64 && tid - 64 < G) lam_mine = p.lamG[(int64_t)a * G + (tid - 64)];
  if (p.ap.done[a]) return;
  const int64_t N = p.N, row = (int64_t)a * N, rowp = (int64_t)a * p.ldw;
  const int sub = (a * p.S + sl) * FAST_NW + wid;               // this warp's list
  unsigned char* stage0 = stream_raw;                                 // FAST_NST stages: v, w0, q, d, 1/d, excl, gid
  uint64_t* bar_full = (uint64_t*)(stream_raw + (size_t)FAST_NST * FAST_STAGE_BYTES);
  uint64_t* bar_empty = bar_full + FAST_NST;
  double* lamS = (double*)(bar_empty + FAST_NST);
  double* scratch = lamS + Gb;                                        // 8 * 32 (CHECK reduction)

  const int64_t i_beg = (int64_t)sl * p.slice_len, i_end = min(N, i_beg + p.slice_len);
  const int nchunk = (int)((i_end - i_beg + FAST_CH - 1) / FAST_CH);
  const uint32_t elem_bytes = 40u + (p.excl ? 1u : 0u) + (G ? 1u : 0u);
  const double* qsrc = p.q ? p.q + rowp : p.mu + row;
  // thread 0: start the copies of chunk c into its stage
  auto issue = [&](int c) {
    const int st = c % FAST_NST;
    const int64_t i0 = i_beg + (int64_t)c * FAST_CH;
    const uint32_t nc = (uint32_t)min((int64_t)FAST_CH, i_end - i0);
    unsigned char* sb = stage0 + (size_t)st * FAST_STAGE_BYTES;
    mbar_expect_tx(&bar_full[st], nc * elem_bytes);
    bulk_g2s(sb, p.v + rowp + i0, nc * 8, &bar_full[st]);
    bulk_g2s(sb + FAST_CH * 8, p.w0 + row + i0, nc * 8, &bar_full[st]);
    bulk_g2s(sb + 2 * FAST_CH * 8, qsrc + i0, nc * 8, &bar_full[st]);
    bulk_g2s(sb + 3 * FAST_CH * 8, p.d + i0, nc * 8, &bar_full[st]);
    bulk_g2s(sb + 4 * FAST_CH * 8, p.invd + i0, nc * 8, &bar_full[st]);
    if (p.excl) bulk_g2s(sb + 5 * FAST_CH * 8, p.excl + row + i0, nc, &bar_full[st]);
    if (G) bulk_g2s(sb + 5 * FAST_CH * 8 + FAST_CH, p.group_id + i0, nc, &bar_full[st]);
  };
  // the first copies start before anything else is read: the account's constants load while they are in flight
  if (tid == 0) {
    for (int st = 0; st < FAST_NST; ++st) { mbar_init(&bar_full[st], 1); mbar_init(&bar_empty[st], FAST_NW); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int c = 0; c < FAST_NST - 1 && c < nchunk; ++c) issue(c);
  }
  if (wid == 1 && lane < 12) cst[lane] = cv;
  if (SB && tid < 4) sbin[tid] = 0ull;
  if (tid >= 64 && tid - 64 < G) lamS[tid - 64] = lam_mine;
  for (int g = tid + FAST_NW * 32 - 64; g < G; g += FAST_NW * 32) lamS[g] = p.lamG[(int64_t)a * G + g];   // (G > 192 only)
  __syncthreads();
  const double lo_a = cst[0], hi_a = cst[1];
  if (!(hi_a - lo_a <= 4.0)) {            // box wider than the fixed-point range of the bins: generic path in k_prox_root
    if (tid == 0 && sl == 0) p.lflag[a] = 1;
    if (lane == 0) { p.lcnt[sub] = 0; p.lcnt[p.A * p.S * FAST_NW + sub] = 0; }
    for (int c = 0; c < FAST_NST - 1 && c < nchunk; ++c) mbar_wait(&bar_full[c], 0u);   // no copy may outlive the CTA
    return;
  }
  const double W = cst[2], Wt = cst[3];
  // Two-level lists: an asset that only the WIDE window (W) can reach but the TIGHT one (Wt, what the thresholds are
  // expected to move by) cannot is finished speculatively as dead - outputs written, trade added to the second set of
  // bins - and parked at the back of the warp's list; k_prox_root looks at those entries only when its solution
  // leaves the tight window.  Check / final launches keep one level (their residual terms must not be speculative).
  const bool split = !CHECK && Wt < 0.125 * W;
  const double Wn = split ? Wt : W;
  const double gam = cst[4], c = cst[5], cg = c * gam, icg = 1.0 / cg;
  const double kappa = cst[6];
  const double lam_b = kappa + cst[7], Delta = lam_b + kappa;
  const double tau = cst[8];
  const double igc = 1.0 / (gam * (1.0 + c));
  double aw = cst[9], bw = cst[10];
  if (!(cst[11] == 1.0 && isfinite(tau))) bw = aw;

  double nx = 0, nz = 0, nrp = 0, nrd = 0, nPx = 0, ny = 0, nq = 0;
  LiveEnt* mylist = p.lraw + (int64_t)sub * p.capw;
  unsigned long long* cbin = p.cbin + (int64_t)a * 2 * Gb;
  const int64_t fbin_off = (int64_t)p.A * 2 * Gb;                       // second set of bins: speculative trades
  const unsigned lt = (1u << lane) - 1u;
  int n = 0, nw_ = 0;
  const double aN_lo = aw - Wn, aN_hi = aw + Wn, bN_lo = bw - Wn - Delta, bN_hi = bw + Wn - Delta;
  const double aW_lo = aw - W, aW_hi = aw + W, bW_lo = bw - W - Delta, bW_hi = bw + W - Delta;
  double* rtp = p.rt + rowp + i_beg + tid;
  double* ccp = p.cc + rowp + i_beg + tid;
  for (int c = 0; c < nchunk; ++c) {
    const int st = c % FAST_NST;
    if (tid == 0 && c + FAST_NST - 1 < nchunk) {          // refill the stage chunk c - 1 lived in
      const int cn = c + FAST_NST - 1;
      if (cn >= FAST_NST) mbar_wait(&bar_empty[cn % FAST_NST], (uint32_t)((cn / FAST_NST - 1) & 1));
      issue(cn);
    }
    mbar_wait(&bar_full[st], (uint32_t)((c / FAST_NST) & 1));
    const unsigned char* sb = stage0 + (size_t)st * FAST_STAGE_BYTES;
    const double* sv = (const double*)sb + tid;
    const unsigned char* sx = sb + 5 * FAST_CH * 8 + tid;
    const int64_t i0 = i_beg + (int64_t)c * FAST_CH;
    const int nc = (int)min((int64_t)FAST_CH, i_end - i0);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int t = tid + h * (FAST_NW * 32);
      const bool valid = t < nc;                                  // (stale stage data beyond nc is read but not used)
      const double v = sv[h * 256];
      const double w0 = sv[FAST_CH + h * 256];
      const double qraw = sv[2 * FAST_CH + h * 256];
      const double rho = cg * sv[3 * FAST_CH + h * 256];
      const double iv = sv[4 * FAST_CH + h * 256];
      const bool ex = p.excl ? sx[h * 256] != 0 : false;
      int g = 0;
      double lg = 0.0;
      if (G) { g = sx[FAST_CH + h * 256]; lg = lamS[g]; }
      const double qm = p.q ? -qraw : qraw;                          // -q_i
      const double u = v - w0;
      const double T = fma(u, rho, -lam_b);
      const double tA = T - lg;
      // Branch-free classification (a warp almost always holds a few excluded / sold-out assets, so a rare-case
      // branch would be taken by nearly every warp).  Inside its box an asset's buy amount is 0 if the buy
      // threshold of the window cannot reach it, the whole room wB if even the far end of the window fills it,
      // and depends on the thresholds (live) in between; the same for the sell side.
      const bool inbox = w0 >= lo_a && w0 <= hi_a;
      const double wB = hi_a - w0, wS = w0 - lo_a;
      const double wBr = wB * rho, wSr = wS * rho;
      const bool b_reach = tA > aN_lo, b_full = tA - aN_hi >= wBr;
      const bool s_reach = tA < bN_hi, s_full = bN_lo - tA >= wSr;
      double bc = (b_reach && b_full) ? wB : 0.0;
      double sc = (s_reach && s_full) ? wS : 0.0;
      bool live = (b_reach && !b_full) || (s_reach && !s_full) || !inbox;   // outside its box (rare): live
      bool spec = false;                                                     // dead in the tight window, live in the wide one
      if (split) spec = !live && ((tA > aW_lo && !(tA - aW_hi >= wBr)) || (tA < bW_hi && !(bW_lo - tA >= wSr)));
      if (ex) { bc = 0.0; sc = w0; live = !(w0 >= 0.0 && w0 <= 4.0); spec = false; }   // lo = hi = 0: the trade is -w0
      live = live && valid;
      spec = spec && valid;
      const double tc = bc - sc;                                             // trade of a dead asset
      const double z = w0 + tc;
      const double rt = fma(rho, (w0 - u) + 2.0 * tc, qm) * (iv * igc);      // (rho (2 z - v) - q) / M_i
      if (valid && !live) {
        rtp[h * 256] = rt;
        ccp[h * 256] = rt - z;
        unsigned long long* bin = SB ? (spec ? sbin + 2 : sbin) : (spec ? cbin + fbin_off : cbin);   // (with groups the bins are spread: direct)
        if (bc > 0.0) atomicAdd(&bin[g], (unsigned long long)__double2ull_rn(bc * PRISM_FIX_SCALE));
        if (sc > 0.0) atomicAdd(&bin[Gb + g], (unsigned long long)__double2ull_rn(sc * PRISM_FIX_SCALE));
        if (CHECK) {
          const int64_t i = i0 + t;
          p.w_out[row + i] = z;            // speculative: kept if the account turns out to have converged
          const double x = p.xs[rowp + i], pq = p.pxq[rowp + i];
          const double y = rho * (v - z);
          nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
          nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq + qm)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qm));
          if (!(x == x) || !(pq == pq) || !(z == z)) nrp = INFINITY;
        }
      }
      const unsigned m = __ballot_sync(0xffffffffu, live);
      const unsigned ms = split ? __ballot_sync(0xffffffffu, spec) : 0u;
      if (m | ms) {
        if (live || spec) {
          LiveEnt e;
          e.T = T; e.w0 = w0; e.ir = iv * icg; e.pad = 0;
          e.meta = (uint32_t)(i0 + t) | ((uint32_t)g << PROX_META_IDX_BITS) | ((uint32_t)(ex ? 1 : (inbox ? 0 : 2)) << 30);
          // tight list from the front, speculative entries from the back of the same buffer (n + nw_ <= capw always)
          mylist[live ? n + __popc(m & lt) : p.capw - 1 - (nw_ + __popc(ms & lt))] = e;
        }
        n += __popc(m);
        nw_ += __popc(ms);
      }
    }
    rtp += FAST_CH; ccp += FAST_CH;
    __syncwarp();
    if (lane == 0) mbar_arrive(&bar_empty[st]);
  }
  if (lane == 0) { p.lcnt[sub] = n; p.lcnt[p.A * p.S * FAST_NW + sub] = nw_; }
  if (SB) {
    __syncthreads();
    if (tid < 4) {
      const unsigned long long x = sbin[tid];
      if (x) atomicAdd(tid < 2 ? &cbin[tid] : &cbin[fbin_off + (tid - 2)], x);
    }
  }
  if (CHECK) {
    double val[7] = {nx, nz, nrp, nrd, nPx, ny, nq};
    block_reduce<7, 1>(val, scratch);
    if (tid < 7) p.chkp[((int64_t)a * p.S + sl) * 8 + tid] = val[tid];
  }
}

// ------------------------------------------------------------------------------------------------ root kernel
// Live-list source: the compacted list of one account in global memory (L2 resident), plus the fixed-point
// totals of the dead assets (cbin: buys [0, Gb), sells [Gb, 2 Gb) per group, in units of 2^-60).
#define ROOT_NSL 4            // sub-lists of a filtered list: one per warp of the root CTA
struct SrcLiveG {
  double lo_a, hi_a;
  const LiveEnt* ent;               // nsl sub-lists, sub-list k at ent + k * stride with cnt[k] entries, visited in order
  int nsl, stride, cnt[ROOT_NSL];
  const unsigned long long* cbin;   // shared memory: fixed-point totals of the assets that are not in the list
  int Gb;
  double cPt, cRt;
  double scale;                     // 1, or the stride of a SAMPLED list (every stride-th live asset stands for stride of them)
  template <int NV, int OP>
  __device__ __forceinline__ void reduce(double (&val)[NV], double* scratch) const { block_reduce<NV, OP>(val, scratch); }
  __device__ __forceinline__ double cP() const { return cPt; }
  __device__ __forceinline__ double cR() const { return cRt; }
  __device__ __forceinline__ double cPg(int g) const { return (double)cbin[g] * PRISM_FIX_INV; }
  __device__ __forceinline__ double cRg(int g) const { return (double)cbin[Gb + g] * PRISM_FIX_INV; }
  __device__ __forceinline__ int64_t decode(const double2& a, const double2& b, ElemConst& e, int& g) const {
    e.T = a.x; e.w0 = a.y; e.ir = b.x;
    const uint32_t m = (uint32_t)__double_as_longlong(b.y);
    const int c = (int)(m >> 30);
    g = (int)((m >> PROX_META_IDX_BITS) & 0xffu);
    if (c == 0) { e.bl = 0.0; e.sl = 0.0; e.wB = hi_a - e.w0; e.wS = e.w0 - lo_a; }
    else elem_ranges(e, c == 1 ? 0.0 : lo_a, c == 1 ? 0.0 : hi_a);
    return (int64_t)(m & ((1u << PROX_META_IDX_BITS) - 1u));
  }
  // long lists (first iterations: every asset is live) are latency-bound: four entries' loads are issued together
  template <class F>
  __device__ __forceinline__ void for_each(F f) const {
    const int nt = blockDim.x;
    for (int k = 0; k < nsl; ++k) {
      const LiveEnt* el = ent + (int64_t)k * stride;
      const int n = cnt[k];
      int j = threadIdx.x;
      for (; j + 3 * nt < n; j += 4 * nt) {
        double2 a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { a[u] = *((const double2*)(el + j + u * nt)); b[u] = *((const double2*)(el + j + u * nt) + 1); }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          ElemConst e; int g;
          const int64_t i = decode(a[u], b[u], e, g);
          f(i, e, g, 0, (const double*)nullptr, (const double*)nullptr);
        }
      }
      for (; j < n; j += nt) {
        const double2 a = *((const double2*)(el + j)), b = *((const double2*)(el + j) + 1);
        ElemConst e; int g;
        const int64_t i = decode(a, b, e, g);
        f(i, e, g, 0, (const double*)nullptr, (const double*)nullptr);
      }
    }
  }
  template <class F>
  __device__ __forceinline__ void for_each_uniform(F f) const {
    for (int k = 0; k < nsl; ++k) {
      const LiveEnt* el = ent + (int64_t)k * stride;
      const int n = cnt[k];
      for (int j0 = 0; j0 < n; j0 += blockDim.x) {
        const int j = j0 + threadIdx.x;
        const bool valid = j < n;
        ElemConst e; int g = 0; int64_t i = 0;
        if (valid) {
          const double2 a = *((const double2*)(el + j)), b = *((const double2*)(el + j) + 1);
          i = decode(a, b, e, g);
        }
        f(valid, i, e, g, 0, (const double*)nullptr, (const double*)nullptr);
      }
    }
  }
};

__host__ __device__ inline size_t root_smem_bytes(int G, int nsub) {
  const int Gb = G > 0 ? G : 1;
  return (size_t)(16 * 32 + ROOT_MAXW * Gb + 6 * Gb + 6 * Gb + 8 + 4 * (Gb + ROOT_MAXW)) * 8 + (size_t)(nsub + 1 + ROOT_MAXW * Gb + 3 * Gb + 16 + ROOT_MAXW + ROOT_NSL) * 4 + 32 + (size_t)ROOT_SCAP * 32;
}

// Sum over the block of terms that only the first `nfront` threads hold (the others pass zeros): with nfront <= 32
// warp 0 alone reduces and publishes - one butterfly and one barrier less than block_reduce on the critical path of
// every pass, and the same bits (block_reduce would add the other warps' zeros).
template <int NV>
__device__ __forceinline__ void front_sum(double (&val)[NV], double* scratch, int nfront) {
  if (nfront > 32) { block_reduce<NV, 0>(val, scratch); return; }
  if (threadIdx.x < 32) {
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      const double x = warp_sum(val[q]);
      if ((threadIdx.x & 31) == 0) scratch[q] = x;
    }
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < NV; ++q) val[q] = scratch[q];
  __syncthreads();      // scratch may be reused by the next call
}

// One pass over the grouped list: per (pseudo-)group q the buys, sells and their slopes at thresholds (al, bd + Delta)
// shifted by the group's multiplier -> gv[4 q .. 4 q + 3].  Warp w owns the groups w, w + nw, ...; fixed order.
// buys, sells and slopes of one list entry at thresholds (a0, b0); the common class (inside its box) without branches
__device__ __forceinline__ void root_entry(const SrcLiveG& src, const double2& ea, const double2& eb, double a0, double b0,
                                           double& sp, double& sr, double& slp, double& slr) {
  const uint32_t m = (uint32_t)__double_as_longlong(eb.y);
  const double T = ea.x, w0 = ea.y, ir = eb.x;
  if ((m >> 30) == 0) {
    const double wB = src.hi_a - w0, wS = w0 - src.lo_a;
    const double tb = (T - a0) * ir, ts = (b0 - T) * ir;
    sp += tb <= 0.0 ? 0.0 : (tb >= wB ? wB : tb);
    sr += ts <= 0.0 ? 0.0 : (ts >= wS ? wS : ts);
    slp += (tb > 0.0 && tb < wB) ? ir : 0.0;
    slr += (ts > 0.0 && ts < wS) ? ir : 0.0;
  } else {
    ElemConst e; int g; double mvb, mvs;
    src.decode(ea, eb, e, g);
    sp += buy_amt(e, a0, mvb); sr += sell_amt<false>(e, b0, nullptr, nullptr, 0, mvs); slp += mvb; slr += mvs;
  }
}
__device__ __forceinline__ void root_pass(const SrcLiveG& src, const int* poff, int ngrp, const double* lamS, int G,
                                          double al, double bd, double* gv) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int q = wid; q < ngrp; q += nw) {
    const double lg = G ? lamS[q] : 0.0;
    const double a0 = al + lg, b0 = bd + lg;
    double sp = 0, sr = 0, slp = 0, slr = 0;
    const int j1 = poff[q + 1];
    int j = poff[q] + lane;
    for (; j + 96 < j1; j += 128) {
      double2 ea[4], eb[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { ea[u] = *((const double2*)(src.ent + j + 32 * u)); eb[u] = *((const double2*)(src.ent + j + 32 * u) + 1); }
#pragma unroll
      for (int u = 0; u < 4; ++u) root_entry(src, ea[u], eb[u], a0, b0, sp, sr, slp, slr);
    }
    for (; j < j1; j += 32) {
      const double2 ea = *((const double2*)(src.ent + j)), eb = *((const double2*)(src.ent + j) + 1);
      root_entry(src, ea, eb, a0, b0, sp, sr, slp, slr);
    }
    sp = warp_sum(sp); sr = warp_sum(sr); slp = warp_sum(slp); slr = warp_sum(slr);
    if (lane == 0) { const double sc = src.scale; gv[4 * q] = sp * sc; gv[4 * q + 1] = sr * sc; gv[4 * q + 2] = slp * sc; gv[4 * q + 3] = slr * sc; }
  }
  __syncthreads();
}

// The grouped list as a source of the nested robust solver prox_rootfind: its evaluation routines are overloaded
// here so that every trial evaluation is one lean root_pass (the per-group sums it leaves in gv also serve the
// selected-group sums and the all-groups pass of the solver).
struct SrcGrouped {
  const SrcLiveG* L;
  const int* poff;
  int ngrp;
  double* gv;
  __device__ __forceinline__ double cP() const { return L->cPt; }
  __device__ __forceinline__ double cR() const { return L->cRt; }
};
template <bool LOTS>
__device__ __noinline__ void prox_eval(const SrcGrouped& s, const double* lamS, int G, double al, double bd, int s1, int s2,
                                       double* scratch, double* out) {
  root_pass(*s.L, s.poff, s.ngrp, lamS, G, al, bd, s.gv);
  double val[4] = {0.0, 0.0, 0.0, 0.0};
  if ((int)threadIdx.x < s.ngrp) {
#pragma unroll
    for (int q = 0; q < 4; ++q) val[q] = s.gv[4 * threadIdx.x + q];
  }
  front_sum<4>(val, scratch, s.ngrp);
  out[0] = val[0] + s.L->cPt; out[1] = val[1] + s.L->cRt; out[2] = val[2]; out[3] = val[3];
#pragma unroll
  for (int q = 4; q < 12; ++q) out[q] = 0.0;
  if (s1 >= 0) { out[4] = s.gv[4 * s1] + s.L->cPg(s1); out[5] = s.gv[4 * s1 + 1] + s.L->cRg(s1); out[6] = s.gv[4 * s1 + 2]; out[7] = s.gv[4 * s1 + 3]; }
  if (s2 >= 0) { out[8] = s.gv[4 * s2] + s.L->cPg(s2); out[9] = s.gv[4 * s2 + 1] + s.L->cRg(s2); out[10] = s.gv[4 * s2 + 2]; out[11] = s.gv[4 * s2 + 3]; }
  __syncthreads();                                       // gv is rewritten by the next pass
}
template <bool LOTS>
__device__ __noinline__ void prox_group_sums(const SrcGrouped& s, const double* lamS, int G, double al, double bd,
                                             const double* gw0, double* gbin, double* gsum) {
  root_pass(*s.L, s.poff, s.ngrp, lamS, G, al, bd, s.gv);
  for (int g = threadIdx.x; g < G; g += blockDim.x)
    gsum[g] = gw0[g] + (s.gv[4 * g] + s.L->cPg(g)) - (s.gv[4 * g + 1] + s.L->cRg(g));
  __syncthreads();
}
template <bool LOTS>
__device__ __noinline__ void prox_brackets(const SrcGrouped& s, double Delta, double* scratch, double* out) {
  prox_brackets<LOTS>(*s.L, Delta, scratch, out);
}
template <bool LOTS>
__device__ __noinline__ void prox_eval_multi(const SrcGrouped& s, const double* lamS, int G, double a0, double da, double b0,
                                             double db, double* scratch, double* outP, double* outR) {
  const SrcLiveG& L = *s.L;
  double sp[PROX_KSEC], sr[PROX_KSEC];
#pragma unroll
  for (int k = 0; k < PROX_KSEC; ++k) { sp[k] = 0.0; sr[k] = 0.0; }
  const int n = L.cnt[0];
  for (int j = threadIdx.x; j < n; j += blockDim.x) {
    const double2 ea = *((const double2*)(L.ent + j)), eb = *((const double2*)(L.ent + j) + 1);
    const uint32_t m = (uint32_t)__double_as_longlong(eb.y);
    const double lg = G ? lamS[(m >> PROX_META_IDX_BITS) & 0xffu] : 0.0;
    if ((m >> 30) == 0) {
      const double T = ea.x, w0 = ea.y, ir = eb.x, wB = L.hi_a - w0, wS = w0 - L.lo_a;
      const double tb0 = (T - a0 - lg) * ir, ts0 = (b0 + lg - T) * ir, dtb = da * ir, dts = db * ir;
#pragma unroll
      for (int k = 0; k < PROX_KSEC; ++k) {
        const double tb = tb0 - k * dtb, ts = ts0 + k * dts;
        sp[k] += tb <= 0.0 ? 0.0 : (tb >= wB ? wB : tb);
        sr[k] += ts <= 0.0 ? 0.0 : (ts >= wS ? wS : ts);
      }
    } else {
      ElemConst e; int g;
      L.decode(ea, eb, e, g);
#pragma unroll
      for (int k = 0; k < PROX_KSEC; ++k) {
        double mvb, mvs;
        sp[k] += buy_amt(e, a0 + k * da + lg, mvb);
        sr[k] += sell_amt<false>(e, b0 + k * db + lg, nullptr, nullptr, 0, mvs);
      }
    }
  }
  block_reduce<PROX_KSEC, 0>(sp, scratch);
  block_reduce<PROX_KSEC, 0>(sr, scratch);
#pragma unroll
  for (int k = 0; k < PROX_KSEC; ++k) { outP[k] = sp[k] * L.scale + L.cPt; outR[k] = sr[k] * L.scale + L.cRt; }
}

template <bool CHECK, int NT>
__global__ void __launch_bounds__(NT, NT <= 128 ? 4 : 1) k_prox_root(const __grid_constant__ ProxArgs p, int mode) {
  extern __shared__ __align__(16) unsigned char root_raw[];
  __shared__ SrcLiveG src;                 // CTA-uniform objects live in shared memory, not on the threads' stacks
  __shared__ SrcGrouped sgrp;
  __shared__ ProxShared sh;
  __shared__ int nback_s;                  // entries at the backs of the lists (speculatively finished by the streaming pass)
  const int a = blockIdx.x;
  if (p.ap.done[a]) return;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nt = blockDim.x, nw = nt >> 5;
  if (tid == 0) nback_s = 0;
  const int G = p.G, Gb = G > 0 ? G : 1;
  const int64_t N = p.N, row = (int64_t)a * N, rowp = (int64_t)a * p.ldw;
  const int nsub = p.S * FAST_NW;
  const int ngrp = G > 0 ? G : nw;                       // without groups: nw slices of the list, for load balance
  double* d0 = (double*)root_raw;
  double* scratch = d0; d0 += 16 * 32;
  double* gbin = d0; d0 += ROOT_MAXW * Gb;               // nw x Gb
  double* lamS = d0; d0 += Gb;
  double* gsum = d0; d0 += Gb;
  double* band_lo = d0; double* band_hi = d0 + Gb; double* gw0 = d0 + 2 * Gb; double* lamW = d0 + 3 * Gb; d0 += 4 * Gb;
  unsigned long long* cbin = (unsigned long long*)d0; d0 += 2 * Gb;    // dead assets of the streaming pass
  unsigned long long* fbin = (unsigned long long*)d0; d0 += 2 * Gb;    // + list entries outside the tight window
  unsigned long long* ubin = (unsigned long long*)d0; d0 += 2 * Gb;    // their sum: what the solve uses
  double* chk = d0; d0 += 8;
  double* gv = d0; d0 += 4 * (Gb + ROOT_MAXW);           // per (pseudo-)group sums of one pass (ngrp <= max(G, nw))
  int* offs = (int*)d0;                                  // 2 nsub + 1: start of raw list k in the sequence of lists in use
  int* wcnt = offs + 2 * nsub + 1;                       // nw x Gb: entries of group g in warp w's part (then running offsets)
  int* goff = wcnt + ROOT_MAXW * Gb;                     // Gb + 1 group offsets of the grouped list
  int* poff = goff + Gb + 1;                             // ngrp + 1 (pseudo-)group offsets used by the passes
  int* act = poff + Gb + ROOT_MAXW + 1;                  // Gb: band state -1 lower active, 0 inactive, +1 upper active
  int* selS = act + Gb;
  LiveEnt* ents = (LiveEnt*)(((uintptr_t)(selS + 4) + 15) & ~(uintptr_t)15);   // ROOT_SCAP entries

  const double gam = p.gamma[a], c = p.ap.c[a], cg = c * gam;
  const double kappa = p.kappa ? p.kappa[a] : 0.0;
  const double lam_b = kappa + (p.c_buy ? p.c_buy[a] : 0.0), Delta = lam_b + kappa;
  const double tau = p.tau ? p.tau[a] : INFINITY;
  const double igc = 1.0 / (gam * (1.0 + c));
  const double W = p.ap.wins[a], Wt = p.ap.win[a];       // window of the streaming pass; tight window (32 x last movement)
  const bool split = !CHECK && Wt < 0.125 * W;           // the streaming pass made two-level lists (same test there)
  const double src_lo = p.lo[a], src_hi = p.hi[a];
  const double b = p.ap.bsum[a];
  double aw = p.ap.alpha[a], bw = p.ap.beta[a];
  int amode_w = p.ap.mode[a];
  if (!(amode_w == 1 && isfinite(tau))) { amode_w = 0; bw = aw; }
  const int generic = p.lflag[a];

  // ---- gather: band data, warm-start multipliers, fixed-point bins (cleared for the next launch)
  for (int g = tid; g < G; g += nt) {
    const int64_t e = (int64_t)a * G + g;
    band_lo[g] = p.band_lo[e]; band_hi[g] = p.band_hi[e]; gw0[g] = p.gw0[e];
    lamW[g] = lamS[g] = p.lamG[e];
  }
  for (int g = tid; g < 2 * Gb; g += nt) {
    unsigned long long* src_bin = p.cbin + (int64_t)a * 2 * Gb + g;
    cbin[g] = *src_bin;
    *src_bin = 0ull;
    src_bin += (int64_t)p.A * 2 * Gb;                    // speculative trades (entries at the back of the lists)
    fbin[g] = *src_bin;
    *src_bin = 0ull;
  }
  for (int e = tid; e < nw * Gb; e += nt) wcnt[e] = 0;
  for (int k = tid; k < nsub; k += nt) offs[k + 1] = p.lcnt[(int64_t)a * nsub + k];
  __syncthreads();
  bool fallback = generic != 0;
  int nlist_used = nsub;
  RootState rs;
  rs.alpha = aw; rs.beta = bw; rs.amode = amode_w; rs.n_eval = 0; rs.capped = 0;
  // band ramp: the first iterations project without the group bands (an exact prox of the relaxed problem); their
  // thresholds still move a lot then and a band solve would be wasted.  Never on check / final launches.
  const bool exact = CHECK || (mode & PROX_FINAL);
  const bool bands_on = G > 0 && (exact || p.iter > p.band_start);
  rs.nobands = bands_on ? 0 : 1;
  // ... and then join gradually: for band_ramp iterations the limits are widened by a slack that shrinks linearly from
  // the largest violation measured at band_start to zero (still an exact prox, of a relaxed problem), so that few bands
  // change state per iteration and the multipliers move in small steps.  Check / final launches never relax.
  if (bands_on && !exact && p.band_ramp > 0 && p.iter < p.band_start + p.band_ramp) {
    const double sl = p.ap.slack[a] * (1.0 - (double)(p.iter - p.band_start) / (double)p.band_ramp);
    for (int g = tid; g < G; g += nt) { band_lo[g] -= sl; band_hi[g] += sl; }
    __syncthreads();
  }
  double mv = 0.0;
  // work areas of the nested solver: set up for BOTH paths (the every-asset path below uses them too)
  if (tid == 0) {
    sh.scratch = scratch; sh.gbin = gbin; sh.lamS = lamS; sh.gsum = gsum; sh.selS = selS;
    sh.band_lo = band_lo; sh.band_hi = band_hi; sh.gw0 = gw0;
    p.lflag[a] = 0;
  }
  __syncthreads();
  if (!fallback) {
    // ---- the raw lists as one sequence (offs = their start offsets); warp w handles a contiguous quarter of it.
    // Level 0: the tight parts (fronts) of the nsub lists.  Level 1 (only after a solution left the tight window):
    // fronts and backs together, 2 nsub lists; entry m of a back sits at position capw - 1 - m of its buffer.
    const unsigned lt = (1u << lane) - 1u;
    const LiveEnt* lr = p.lraw + (int64_t)a * nsub * p.capw;
    const int32_t* lcw = p.lcnt + (int64_t)p.A * nsub + (int64_t)a * nsub;   // lengths of the backs
    int nlist = nsub, nraw = 0, j_beg = 0, j_end = 0;
    // Sampled root find (prism_settings.sample_until): plain launches of the first iterations, while the bands are still
    // out of the projection, solve for the thresholds on every stride-th live asset (each standing for stride of them,
    // stride such that the sample fits the shared-memory list) and apply them to all: an inexact prox where exactness buys
    // nothing - every asset is still live then and an exact solve walks the 9,800-entry lists 7-24 times.
    const bool sampm = !exact && !bands_on && p.iter < p.sample_until;
    int stride = 1;
    auto scan_lists = [&](int level) {
      nlist = level ? 2 * nsub : nsub;
      __syncthreads();
      for (int k = tid; k < nlist; k += nt) offs[k + 1] = k < nsub ? p.lcnt[(int64_t)a * nsub + k] : lcw[k - nsub];
      __syncthreads();
      if (wid == 0) {                                      // inclusive scan of the list lengths
        int carry = 0;
        for (int k0 = 0; k0 < nlist; k0 += 32) {
          int v = k0 + lane < nlist ? offs[k0 + lane + 1] : 0;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += t; }
          if (k0 + lane < nlist) offs[k0 + lane + 1] = v + carry;
          carry += __shfl_sync(0xffffffffu, v, 31);
        }
        if (lane == 0) offs[0] = 0;
      }
      __syncthreads();
      nraw = offs[nlist];
      stride = (sampm && nraw > ROOT_SCAP) ? (nraw + ROOT_SCAP - 1) / ROOT_SCAP : 1;
      const int nsmp = (nraw + stride - 1) / stride;       // the sort and the solve see samples j = 0 .. nsmp - 1 (entry j * stride)
      const int segw = (((nsmp + nw - 1) / nw) + 31) & ~31;
      j_beg = min(nsmp, wid * segw); j_end = min(nsmp, (wid + 1) * segw);
    };
    // entry j of the sequence; a thread asks for ascending j, so the list is found by advancing a cursor (cur: the list the
    // previous entry sat in; start it at 0) instead of a binary search per entry (12% of the kernel's stall samples in the
    // first iterations went into those searches)
    auto locate = [&](int j, int& cur) -> const LiveEnt* {
      while (cur + 1 < nlist && offs[cur + 1] <= j) ++cur;
      const int pos = j - offs[cur];
      return cur < nsub ? lr + (int64_t)cur * p.capw + pos : lr + (int64_t)(cur - nsub) * p.capw + (p.capw - 1 - pos);
    };
    // ---- group sort (counting sort, stable in sequence order => deterministic): entries -> lcomp (or shared memory) by
    // group.  use_f: the speculative trades of the backs (fbin) count as constants (level 0 of a two-level list).
    auto sort_lists = [&](bool use_f) {
      for (int e = tid; e < nw * Gb; e += nt) wcnt[e] = 0;
      __syncthreads();
      if (!G) { if (lane == 0) wcnt[wid] = j_end - j_beg; }
      else {
        int cur = 0;
        for (int j0 = j_beg; j0 < j_end; j0 += 128) {     // four groups of 32 entries: their loads are issued together
          int g4[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int j = j0 + 32 * u + lane;
            g4[u] = 0x100 + lane;
            if (j < j_end) g4[u] = (int)((__ldg(&locate(j * stride, cur)->meta) >> PROX_META_IDX_BITS) & 0xffu);
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int g = g4[u];
            const unsigned m = __match_any_sync(0xffffffffu, g);
            if (g < 0x100 && lane == __ffs(m) - 1) wcnt[wid * Gb + g] += __popc(m);
            __syncwarp();
          }
        }
      }
      __syncthreads();
      for (int g = tid; g < Gb; g += nt) {               // start of warp w's entries inside group g; group totals
        int run = 0;
        for (int w = 0; w < nw; ++w) { const int t = wcnt[w * Gb + g]; wcnt[w * Gb + g] = run; run += t; }
        goff[g + 1] = run;
      }
      for (int g = tid; g < 2 * Gb; g += nt) ubin[g] = cbin[g] + (use_f ? fbin[g] : 0ull);
      __syncthreads();
      if (tid == 0) {
        goff[0] = 0;
        for (int g = 0; g < Gb; ++g) goff[g + 1] += goff[g];
        const int n = goff[Gb];
        if (G) for (int g = 0; g <= G; ++g) poff[g] = goff[g];
        else for (int q = 0; q <= nw; ++q) poff[q] = (int)((int64_t)n * q / nw);
        unsigned long long sp = 0ull, sr = 0ull;
        for (int g = 0; g < Gb; ++g) { sp += ubin[g]; sr += ubin[Gb + g]; }
        src.lo_a = src_lo; src.hi_a = src_hi; src.ent = n <= ROOT_SCAP ? ents : p.lcomp + (int64_t)a * p.ldc; src.nsl = 1; src.stride = 0; src.cnt[0] = n;
        src.cbin = ubin; src.Gb = Gb; src.cPt = (double)sp * PRISM_FIX_INV; src.cRt = (double)sr * PRISM_FIX_INV;
        src.scale = (double)stride;
      }
      __syncthreads();
      LiveEnt* dst = const_cast<LiveEnt*>(src.ent);
      int cur = 0;
      for (int j0 = j_beg; j0 < j_end; j0 += 128) {
        double2 ea[4], eb[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int j = j0 + 32 * u + lane;
          ea[u] = make_double2(0, 0); eb[u] = make_double2(0, 0);
          if (j < j_end) { const LiveEnt* e = locate(j * stride, cur); ea[u] = __ldg((const double2*)e); eb[u] = __ldg((const double2*)e + 1); }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int j = j0 + 32 * u + lane;
          int g = 0x100 + lane;
          if (j < j_end) g = G ? (int)(((uint32_t)__double_as_longlong(eb[u].y) >> PROX_META_IDX_BITS) & 0xffu) : 0;
          const unsigned m = __match_any_sync(0xffffffffu, g);
          if (g < 0x100) {
            double2* o = (double2*)(dst + goff[g] + wcnt[wid * Gb + g] + __popc(m & lt));
            o[0] = ea[u]; o[1] = eb[u];
          }
          __syncwarp();
          if (g < 0x100 && lane == __ffs(m) - 1) wcnt[wid * Gb + g] += __popc(m);
          __syncwarp();
        }
      }
      __syncthreads();
    };
    // A long list is first solved on its tight part; a solution that leaves the tight window repeats the solve on the
    // whole list, and one that leaves the streaming pass's window sends the account to the generic path.
    double Wf = split ? Wt : INFINITY;
    {
      int nb = 0;
      for (int k = tid; k < nsub; k += nt) nb += lcw[k];
      if (nb) atomicAdd(&nback_s, nb);
    }
    for (int att = 0; att < 2; ++att) {
      scan_lists(att);                                   // level 0: the fronts; level 1: fronts and backs
      nlist_used = nlist;
      sort_lists(split && att == 0);
      rs.alpha = aw; rs.beta = bw; rs.amode = amode_w; rs.capped = 0;
      for (int g = tid; g < G; g += nt) lamS[g] = lamW[g];
      __syncthreads();
      // ---- semismooth Newton on (alpha, beta, lambda_g of the active bands) jointly: one pass over the list per step.
      // The equations are piecewise linear (see prox.cuh): P(alpha, lambda) = (tau + b)/2 and R(beta, lambda) = (tau - b)/2
      // with the cap active, P - R = b with alpha = beta otherwise, and S_g = bound_g for every active band.  Eliminating
      // d lambda_g = (F_g - sP_g d alpha - sR_g d beta) / (sP_g + sR_g) leaves a 2 x 2 system.  Bands enter the active set
      // when violated and leave it when their multiplier changes sign.  Anything irregular (singular step, no convergence
      // in 16 passes) falls back to the nested robust solver prox_rootfind on the same list.
      const double tol = 2e-15 * fmax(1.0, fabs(b) + (isfinite(tau) ? tau : 0.0));
      const double Pt = 0.5 * (tau + b), Rt = 0.5 * (tau - b);
      const double cPt = src.cPt, cRt = src.cRt;
      double al = aw, be = bw;
      int amode = amode_w;
      bool ok = false;
      // Newton iteration; where it fails the nested robust solver; where that runs out of Gauss-Seidel rounds over the
      // bands (it converges linearly when several bands interact) the Newton iteration once more from its state, which is
      // close by then (tr = 1); if that fails too, the robust solver from the warm start with as many rounds as it needs
      // (never from the state a failed Newton iteration leaves: see DESIGN.md, readings: robust root find).
      for (int tr = 0; tr < 2; ++tr) {
      ok = false;
      for (int g = tid; g < G; g += nt) act[g] = lamS[g] > 0.0 ? 1 : (lamS[g] < 0.0 ? -1 : 0);
      __syncthreads();
      for (int itn = 0; itn < 16; ++itn) {
        root_pass(src, poff, ngrp, lamS, G, al, be - Delta, gv);
        ++rs.n_eval;
        // thread q: the terms of (pseudo-)group q; fixed-order block reduction (deterministic)
        double P, R, sP, sR, sA, sB, sAB, rA, rB, sT, sF;
        bool gconv, sing;
        {
          double v16[16];
  #pragma unroll
          for (int q = 0; q < 16; ++q) v16[q] = 0.0;
          if (tid < ngrp) { v16[0] = gv[4 * tid]; v16[1] = gv[4 * tid + 1]; v16[2] = gv[4 * tid + 2]; v16[3] = gv[4 * tid + 3]; }
          if (tid < G) {
            const int g = tid;
            const double pa = v16[2], ra = v16[3], t = pa + ra;
            const double Sg = gw0[g] + (v16[0] + (double)ubin[g] * PRISM_FIX_INV) - (v16[1] + (double)ubin[Gb + g] * PRISM_FIX_INV);
            int ac = act[g];
            if (ac == 0 && bands_on) {
              if (Sg > band_hi[g] + 8.0 * tol) ac = 1; else if (Sg < band_lo[g] - 8.0 * tol) ac = -1;
              if (ac) v16[11] = 1.0;
            }
            if (ac) {
              const double Fg = Sg - (ac > 0 ? band_hi[g] : band_lo[g]);
              if (fabs(Fg) > tol) v16[11] = 1.0;
              if (t > 0.0) { v16[4] = pa * pa / t; v16[5] = ra * ra / t; v16[6] = pa * ra / t; v16[7] = pa * Fg / t; v16[8] = ra * Fg / t; v16[9] = t; v16[10] = Fg; }
              else if (fabs(Fg) > tol) v16[12] = 1.0;
            }
            gsum[g] = Sg;
          }
          front_sum<16>(v16, scratch, ngrp > G ? ngrp : G);
          P = cPt + v16[0]; R = cRt + v16[1]; sP = v16[2]; sR = v16[3];
          sA = v16[4]; sB = v16[5]; sAB = v16[6]; rA = v16[7]; rB = v16[8]; sT = v16[9]; sF = v16[10];
          gconv = !(v16[11] > 0.0); sing = v16[12] > 0.0;
        }
        const double FA = amode == 1 ? P - Pt : P - R - b, FB = amode == 1 ? R - Rt : 0.0;
        if (fabs(FA) <= tol && fabs(FB) <= tol && gconv) {
          if (amode == 1) { if (al >= be) { ok = true; break; } amode = 0; al = be = 0.5 * (al + be); __syncthreads(); continue; }
          if (!isfinite(tau) || P + R <= tau + tol) { ok = true; break; }
          amode = 1; be = al;
          __syncthreads();
          continue;
        }
        if (sing) break;
        double dal, dbe;
        if (amode == 1) {
          const double M11 = -sP + sA, M12 = sAB, M21 = -sAB, M22 = sR - sB, r1 = -FA + rA, r2 = -FB - rB;
          const double det = M11 * M22 - M12 * M21;
          if (fabs(det) > 1e-300) { dal = (r1 * M22 - M12 * r2) / det; dbe = (M11 * r2 - M21 * r1) / det; }
          else if (fabs(r1) <= tol && fabs(M11) <= 1e-300 && fabs(M22) > 1e-300) { dal = 0.0; dbe = r2 / M22; }   // buy side flat and satisfied
          else if (fabs(r2) <= tol && fabs(M22) <= 1e-300 && fabs(M11) > 1e-300) { dbe = 0.0; dal = r1 / M11; }   // sell side flat and satisfied
          else break;
        } else {
          const double den = (sP + sR) - sT;
          if (!(den > 1e-300)) break;
          dal = dbe = (FA - sF) / den;
        }
        if (!(dal == dal) || !(dbe == dbe)) break;
        __syncthreads();
        for (int g = tid; g < G; g += nt) {                // multipliers and active set (thread g owns band g)
          const double pa = gv[4 * g + 2], ra = gv[4 * g + 3], t = pa + ra;
          int ac = act[g];
          const bool was = ac != 0;
          if (!was && bands_on) { if (gsum[g] > band_hi[g] + 8.0 * tol) ac = 1; else if (gsum[g] < band_lo[g] - 8.0 * tol) ac = -1; }
          if (ac && t > 0.0) {
            const double Fg = gsum[g] - (ac > 0 ? band_hi[g] : band_lo[g]);
            double ln = lamS[g] + (Fg - pa * dal - ra * dbe) / t;
            if (!(ln * ac > 0.0)) { ln = 0.0; ac = 0; }     // the multiplier would change sign: the band goes inactive
            lamS[g] = ln;
          }
          act[g] = ac;
        }
        al += dal; be += dbe;
        __syncthreads();
      }
      if (ok) { rs.alpha = al; rs.beta = be; rs.amode = amode; rs.capped = 0; break; }
      {
        // nested robust solver on the same grouped list (lean passes through the SrcGrouped overloads)
        // (it continues from where the Newton iteration stopped when that state is usable)
        // (not with an infinite window while bands are in play - the launch in which they join: the multipliers a failed
        // Newton iteration leaves there can be far off, and the Gauss-Seidel rounds of the robust solver then crawl:
        // 12,000 passes for one account of configs[2] seed 1, minutes for seed 3)
        const bool keep = tr > 0 ? false
                                 : (al == al && be == be && fabs(al - aw) <= 0.5 * W && fabs(be - bw) <= 0.5 * W && (W < INFINITY || !bands_on));
        __syncthreads();
        if (!keep) for (int g = tid; g < G; g += nt) lamS[g] = lamW[g];
        if (tid == 0) { sgrp.L = &src; sgrp.poff = poff; sgrp.ngrp = ngrp; sgrp.gv = gv; }
        __syncthreads();
        rs.alpha = keep ? al : aw; rs.beta = keep ? be : bw; rs.amode = keep ? amode : amode_w;
        rs.max_rounds = (bands_on && tr < 1) ? 2 * G + 2 : (1 << 30);
        prox_rootfind<false>(p, sgrp, a, b, tau, Delta, sh, rs);
        if (rs.capped != 2) break;
        al = rs.alpha; be = rs.beta; amode = rs.amode;
      }
      }
      double mv_l = 0.0;
      for (int g = 0; g < G; ++g) mv_l = fmax(mv_l, fabs(lamS[g] - lamW[g]));
      mv = fmax(fmax(fabs(rs.alpha - aw), fabs(rs.beta - bw)), mv_l);
      if (stride > 1 || mv <= 0.5 * fmin(Wf, W)) break;     // (a sampled solve is inexact by design: no second level, no every-asset path)
      if (!(Wf < INFINITY)) { fallback = true; break; }   // left the streaming window (or NaN): the dead assets were misjudged
      Wf = INFINITY;
      __syncthreads();
    }
    if (!fallback && G > 0 && !exact && p.iter == p.band_start) {   // band ramp: how far outside its bands is this projection?
      __syncthreads();
      root_pass(src, poff, ngrp, lamS, G, rs.alpha, rs.beta - Delta, gv);
      if (tid < 32) {
        double viol = 0.0;
        for (int g = tid; g < G; g += 32) {
          const double Sg = gw0[g] + (gv[4 * g] + (double)ubin[g] * PRISM_FIX_INV) - (gv[4 * g + 1] + (double)ubin[Gb + g] * PRISM_FIX_INV);
          viol = fmax(viol, fmax(Sg - band_hi[g], band_lo[g] - Sg));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) viol = fmax(viol, __shfl_xor_sync(0xffffffffu, viol, o));
        if (tid == 0) p.ap.slack[a] = fmax(viol, 0.0);
      }
      __syncthreads();
    }
  }
  int finished = 0;
  if (!fallback) {
    // ---------------------------------------------------------------- live assets: output (+ residual terms)
    const double alpha = rs.alpha, beta = rs.beta, bdf = beta - Delta;
    const int nlist_o = nlist_used, nraw_all = offs[nlist_o];
    double nx = 0, nz = 0, nrp = 0, nrd = 0, nPx = 0, ny = 0, nq = 0;
    // every entry of the lists the solve used (the others are finished).  Latency-bound (entry -> asset index -> d, q):
    // the loads of four entries, then of their four (d, q) pairs, are issued together.
    int lo = 0;                                          // cursor over the lists (the thread's j ascends)
    for (int j0 = tid; j0 < nraw_all; j0 += 4 * nt) {
      double2 ea4[4], eb4[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int j = j0 + u * nt;
        ea4[u] = make_double2(0.0, 0.0); eb4[u] = make_double2(0.0, 0.0);
        if (j < nraw_all) {
          while (lo + 1 < nlist_o && offs[lo + 1] <= j) ++lo;
          const int pos = j - offs[lo];
          const LiveEnt* ep = p.lraw + (int64_t)a * nsub * p.capw +
                              (lo < nsub ? (int64_t)lo * p.capw + pos : (int64_t)(lo - nsub) * p.capw + (p.capw - 1 - pos));
          ea4[u] = __ldg((const double2*)ep); eb4[u] = __ldg((const double2*)ep + 1);
        }
      }
      double d4[4], q4[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int64_t i = (int64_t)((uint32_t)__double_as_longlong(eb4[u].y) & ((1u << PROX_META_IDX_BITS) - 1u));
        d4[u] = 0.0; q4[u] = 0.0;
        if (j0 + u * nt < nraw_all) { d4[u] = p.d[i]; q4[u] = p.q ? p.q[rowp + i] : -p.mu[row + i]; }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (j0 + u * nt >= nraw_all) continue;
        ElemConst e; int g; double mvb, mvs;
        const int64_t i = src.decode(ea4[u], eb4[u], e, g);
        const double lg = G ? lamS[g] : 0.0;
        const double tr = buy_amt(e, alpha + lg, mvb) - sell_amt<false>(e, bdf + lg, nullptr, nullptr, 0, mvs);
        const double z = e.w0 + tr;
        const double rho = cg * d4[u];
        const double y = e.T + lam_b - tr * rho;
        const double qi = q4[u];
        const double r = rho * z - y - qi;
        const double rt = r * (e.ir * cg) * igc;
        p.rt[rowp + i] = rt;
        p.cc[rowp + i] = rt - z;
        if (CHECK) {
          p.w_out[row + i] = z;
          const double x = p.xs[rowp + i], pq = p.pxq[rowp + i];
          nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
          nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq - qi)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qi));
          if (!(z == z) || !(x == x) || !(pq == pq)) nrp = INFINITY;
        }
      }
    }
    if (CHECK && !(mode & PROX_FINAL)) {
      if (tid < 7) {                                     // residual terms of the dead assets, per slice
        double m = 0.0;
        for (int s = 0; s < p.S; ++s) m = fmax(m, p.chkp[((int64_t)a * p.S + s) * 8 + tid]);
        chk[tid] = m;
      }
      double val[7] = {nx, nz, nrp, nrd, nPx, ny, nq};
      block_reduce<7, 1>(val, scratch);                  // (its barrier also publishes chk)
#pragma unroll
      for (int q = 0; q < 7; ++q) val[q] = fmax(val[q], chk[q]);
      const double rp = val[2] / fmax(fmax(val[0], val[1]), 1e-300);
      const double rd = val[3] / fmax(fmax(val[4], fmax(val[5], val[6])), 1e-300);
      const bool conv = val[2] <= p.eps_abs + p.eps * fmax(val[0], val[1]) && val[3] <= p.eps_abs + p.eps * fmax(val[4], fmax(val[5], val[6])) &&
                        !rs.capped;                                          // never certify on an unfinished root find
      if (!(rp < INFINITY) || !(rd < INFINITY)) fallback = true;             // NaN / Inf: the generic path classifies it
      else if (!conv && p.adapt && p.iter >= p.adapt_start && p.iter - p.ap.nadapt[a] >= p.adapt_every) {
        // H7: rho <- rho sqrt(r_p / r_d), clipped, when the two scaled residuals are out of balance.  The thresholds found
        // above stay valid (they belong to the old rho); every asset's v, r~ and c are rewritten for the new rho by
        // k_prox_rescale right after this kernel (one streaming pass instead of the every-asset path: 10-40 ms per event
        // on configs[4]), and k_factor adopts c_new.
        const double ratio = sqrt(rp / fmax(rd, 1e-300));
        if (tid == 0) {
          if (ratio > 3.0 || ratio < 1.0 / 3.0) { p.ap.c_new[a] = c * fmin(fmax(ratio, 0.2), 5.0); p.ap.refactor[a] = 2; }
          p.ap.nadapt[a] = p.iter;
        }
      }
      if (!fallback) {
        finished = conv ? 1 : 0;
        if (tid == 0) {
          p.resid[(int64_t)a * PRISM_NRES + PRISM_R_PRIMAL] = rp;
          p.resid[(int64_t)a * PRISM_NRES + PRISM_R_DUAL] = rd;
          if (conv) p.ap.conv[a] = 1;
        }
      }
    }
  }
  if (!fallback) {
    // ---------------------------------------------------------------- commit the account's state
    if (mode & PROX_FINAL) finished = 1;                 // (CHECK instantiation: w_out holds z)
    const double alpha = rs.alpha, beta = rs.beta;
    for (int g = tid; g < G; g += nt) p.lamG[(int64_t)a * G + g] = lamS[g];
    if (tid == 0) {
      p.ap.alpha[a] = alpha; p.ap.beta[a] = beta; p.ap.mode[a] = rs.amode;
      // next window of the streaming pass: a multiple of the last movement, never shrunk while its list is short
      // (a wide window then costs nothing and the solution almost never leaves it); infinite for the first iterations
      double Ws = p.win_ratio * next_window(p, alpha, beta, mv);
      const int nl = offs[nlist_used] + (nlist_used == nsub ? nback_s : 0);   // live assets of the streaming window
      if (nl < 256) Ws = fmax(Ws, nl < 64 ? 2.0 * W : W);
      // ... and for the launch in which the group bands join (band ramp): the thresholds jump then, a finite window
      // would send the accounts whose bands bind through the every-asset path
      const bool wide_next = p.iter < 2 || (G > 0 && p.iter == p.band_start && p.band_wide);
      if (wide_next) Ws = INFINITY;
      p.ap.win[a] = wide_next ? INFINITY : next_window(p, alpha, beta, mv); p.ap.wins[a] = Ws;
      if (finished) {                                    // H6: w_out already holds z
        p.ap.done[a] = 1; p.ap.iters[a] = p.iter;
        atomicAdd(&p.counters[0], 1);
        double* du = p.duals + (int64_t)a * PRISM_NDUAL(G);
        du[0] = 0.5 * (alpha + beta);
        du[1] = 0.5 * (alpha - beta);
        for (int g = 0; g < G; ++g) { du[2 + g] = fmax(lamS[g], 0.0); du[2 + G + g] = fmax(-lamS[g], 0.0); }
        p.resid[(int64_t)a * PRISM_NRES + PRISM_R_RHO] = c;
      }
    }
    return;
  }
  // ------------------------------------------------------------------ generic path: every asset, from global memory
  __syncthreads();
  SrcGlobal<false> gsrc(p, a, cg, p.lo[a], p.hi[a], lam_b);
  ProxShared shg = sh;
  prox_body<false>(p, mode | (CHECK ? PROX_CHECK : 0), gsrc, a, gam, c, kappa, lam_b, shg, false);
  if (tid == 0) p.ap.wins[a] = p.win_ratio * p.ap.win[a];
}

// ------------------------------------------------------------------------------------------------ rho change
// Accounts for which the check decided a new rho scale (refactor == 2, c_new): with the thresholds of this launch (exact
// for every asset, live or not: z_i is a closed form of T_i and the thresholds) the carried state is re-expressed,
// v' = z + y / rho_new with y = rho_old (v - z), and r~ = M_new^-1 (rho_new z - y - q), c = r~ - z are rewritten.
// grid = (ceil(N / RESCALE_PER_CTA), accounts); exits at once for every other account.
#define RESCALE_PER_CTA 4096
__global__ void __launch_bounds__(256) k_prox_rescale(const __grid_constant__ ProxArgs p) {
  __shared__ double lamS[PRISM_MAX_GROUPS];
  const int a = blockIdx.y;
  if (p.ap.done[a] || p.ap.refactor[a] != 2) return;
  const int tid = threadIdx.x, G = p.G;
  for (int g = tid; g < G; g += blockDim.x) lamS[g] = p.lamG[(int64_t)a * G + g];
  __syncthreads();
  const int64_t N = p.N, row = (int64_t)a * N, rowp = (int64_t)a * p.ldw;
  const double gam = p.gamma[a], c = p.ap.c[a], cn = p.ap.c_new[a], cg = c * gam, icg = 1.0 / cg, cgn = cn * gam, icgn = 1.0 / cgn;
  const double igc = 1.0 / (gam * (1.0 + cn));
  const double kappa = p.kappa ? p.kappa[a] : 0.0, lam_b = kappa + (p.c_buy ? p.c_buy[a] : 0.0), Delta = lam_b + kappa;
  const double tau = p.tau ? p.tau[a] : INFINITY;
  const double alpha = p.ap.alpha[a];
  const double beta = (p.ap.mode[a] == 1 && isfinite(tau)) ? p.ap.beta[a] : alpha;
  const double lo_a = p.lo[a], hi_a = p.hi[a], bdf = beta - Delta;
  const int64_t i0 = (int64_t)blockIdx.x * RESCALE_PER_CTA, i1 = min(N, i0 + RESCALE_PER_CTA);
  for (int64_t i = i0 + tid; i < i1; i += blockDim.x) {
    const double iv = p.invd[i], di = p.d[i];
    ElemConst e;
    e.w0 = p.w0[row + i];
    const double v = p.v[rowp + i];
    e.T = (v - e.w0) * (cg * di) - lam_b;
    e.ir = iv * icg;
    const bool ex = p.excl && p.excl[row + i];
    elem_ranges(e, ex ? 0.0 : lo_a, ex ? 0.0 : hi_a);
    const double lg = G ? lamS[p.group_id[i]] : 0.0;
    double mvb, mvs;
    const double tr = buy_amt(e, alpha + lg, mvb) - sell_amt<false>(e, bdf + lg, nullptr, nullptr, 0, mvs);
    const double z = e.w0 + tr;
    const double y = e.T + lam_b - tr * (cg * di);         // rho_old (v - z)
    const double qi = p.q ? p.q[rowp + i] : -p.mu[row + i];
    p.v[rowp + i] = z + y * iv * icgn;
    const double rt = (cgn * di * z - y - qi) * iv * igc;  // M_i = gamma d_i (1 + c_new)
    p.rt[rowp + i] = rt;
    p.cc[rowp + i] = rt - z;
  }
}
