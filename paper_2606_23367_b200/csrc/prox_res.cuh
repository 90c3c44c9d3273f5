// prox_res.cuh - the cluster-resident form of the fused proximal / projection step: ONE kernel
// per iteration, one thread-block CLUSTER per account.
//
// The account's assets are cut into C contiguous slices, one per CTA of the cluster (C = 1, 2, 4, 8 or 16, the smallest
// for which a slice fits the shared-memory budget).  Each CTA
//   A. streams its slice once (v, w0, mu, exclusion mask; d, 1/d, group id of the shared universe), keeps
//      T_i = rho_i (v_i - w0_i) - (kappa + c_buy) and w0_i RESIDENT in shared memory (19 bytes per asset) and classifies
//      every asset against the window around the warm-start thresholds: a "dead" asset (buy and sell amounts constant
//      for every threshold inside the window: on the kink, clamped at a bound, excluded) is FINISHED on the spot -
//      r~ = M^-1 r and c = r~ - z written, residual terms accumulated, constant trade added to its group's constants -
//      the others go to a live list (one touch per asset: this pass is what the kernel's instruction count is);
//   B. takes part in the root find for (alpha, beta, lambda_g) of prox.cuh: every trial evaluation is a pass over the
//      live lists of all C slices out of shared memory, the partial sums meet through DISTRIBUTED shared memory
//      (st.shared::cluster into every peer's inbox + one cluster barrier) and are added in rank order, so every CTA
//      holds bit-identical sums and runs the identical (redundant) scalar logic: a joint semismooth Newton iteration,
//      with the nested bracketed solver prox_rootfind as the robust fallback;
//   C. writes the outputs of its live assets at the final thresholds, and on check launches finishes the residual terms,
//      the convergence mask (H6), the rho adaptation (H7) and the returned weights.
// A solution that leaves the window (or a rho change) rebuilds the live list from the resident slice, repeats B and
// rewrites every asset of the slice from shared memory: nothing falls back to another kernel.  Compared with the
// streaming pair k_prox_stream + k_prox_root (prox_fast.cuh) there are no live lists in global memory, no sort, no
// fixed-point bins and no second launch.  All sums are fp64 in a fixed order (deterministic).
// Tax lots and per-asset caps are handled by the same kernel (template LOTS): lot rows are read from global memory for
// live assets only.
#pragma once
#include "prox.cuh"

#define RES_NT 256                 // threads per CTA (two CTAs per SM at <= 128 registers)
#define RES_NW (RES_NT / 32)
#define RES_NV 16                  // widest cluster-wide reduction (values per call)
#define RES_SMEM_BUDGET (112 * 1024)   // dynamic shared memory per CTA: two CTAs per SM
#define RES_IRC 32                 // live entries per warp whose 1 / rho is cached in shared memory
#define RES_U 4                    // assets per thread whose loads are issued together (memory-level parallelism)

__device__ __forceinline__ uint32_t res_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t res_cta_rank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void res_cluster_barrier() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// store v at the address `local` has in the shared memory of CTA `rank` of this cluster
__device__ __forceinline__ void res_store_peer(double* local, uint32_t rank, double v) {
  uint32_t ra;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(res_smem_u32(local)), "r"(rank));
  asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(ra), "d"(v) : "memory");
}

__device__ __forceinline__ void res_mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(res_smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void res_mbar_expect(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(res_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void res_mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok = 0;
  const uint32_t addr = res_smem_u32(bar);
  while (!ok) {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
  }
}
// bulk copy (TMA engine, 1-D) global -> this CTA's shared memory; bytes and both addresses multiples of 16
__device__ __forceinline__ void res_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(res_smem_u32(dst)), "l"(src), "r"(bytes), "r"(res_smem_u32(bar)) : "memory");
}

// lanes holding the same group are summed in ascending lane order, the lowest lane adds the sums to this warp's bins
// bins[NQ * g + q] (deterministic; call from warp-uniform control flow)
// single: the problem has one (pseudo-)group (G = 0): the warp's terms are summed by a fixed butterfly instead - five
// steps, not one per contributing lane (the serial form was 12% of this kernel's stall samples on configs[1])
template <int NQ>
__device__ __forceinline__ void res_group_add(double* bins, int g, const double (&x)[NQ], bool valid, bool single = false) {
  const int lane = threadIdx.x & 31;
  if (single) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      double y = valid ? x[q] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) y += __shfl_xor_sync(0xffffffffu, y, o);
      if (lane == 0) bins[q] += y;
    }
    __syncwarp();
    return;
  }
  const int key = valid ? g : (0x40000000 + lane);
  const unsigned m = __match_any_sync(0xffffffffu, key);
  unsigned rem = m;
  double s[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) s[q] = 0.0;
  while (__any_sync(0xffffffffu, rem != 0u)) {
    const int src = rem ? (__ffs(rem) - 1) : lane;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      const double y = __shfl_sync(0xffffffffu, x[q], src);
      if (rem) s[q] += y;
    }
    if (rem) rem &= rem - 1u;
  }
  if (valid && lane == __ffs(m) - 1) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) bins[NQ * g + q] += s[q];
  }
  __syncwarp();
}

// Shared-memory footprint of one CTA for a slice of SL assets (host and device agree on it through this function).
struct ResLayout {
  size_t Ts, ws, live, meta, irc, inbox, ginbox, gbin, wpart, grp, nst, seq, lcnt, mbar, bytes;
};
__host__ __device__ inline ResLayout res_layout(int SL, int G, int C) {
  const size_t Gb = G > 0 ? G : 1;
  ResLayout L;
  size_t o = 0;
  L.Ts = o; o += (size_t)SL * 8;
  L.ws = o; o += (size_t)SL * 8;
  L.inbox = o; o += (size_t)2 * C * RES_NV * 8;           // [2][C][RES_NV]   cluster-wide scalar reductions
  L.ginbox = o; o += (size_t)2 * C * 4 * Gb * 8;          // [2][C][4 Gb]     cluster-wide per-group sums
  L.gbin = o; o += (size_t)RES_NW * 4 * Gb * 8;           // [NW][4 Gb]       per-warp group bins
  L.wpart = o; o += (size_t)RES_NW * RES_NV * 8;          // [NW][RES_NV]     per-warp partials
  L.grp = o; o += (size_t)9 * Gb * 8 + 32;                // lamS lamW band_lo band_hi gw0 gsum cPg cRg, act + sel (ints)
  L.nst = o; o += (size_t)16 * 8;                         // Newton state published by warp 0; dummy work area
  L.irc = o; o += (size_t)RES_NW * RES_IRC * 8;           // 1 / rho of the first RES_IRC live entries of every warp
  L.mbar = o; o += 16;                                    // mbarrier of the bulk copies
  L.seq = o; o += (size_t)RES_NT * 4;                     // per-thread reduction counters (inbox parity)
  L.lcnt = o; o += (size_t)RES_NW * 4;
  L.live = o; o += (size_t)SL * 2;
  L.meta = o; o += (size_t)SL;                            // bits 0-5 group, bit 6 excluded
  L.bytes = (o + 15) & ~(size_t)15;
  return L;
}
__host__ __device__ inline bool res_fits(int64_t N, int G, int C, int* SL_out) {
  int64_t per = (N + C - 1) / C;
  per = (per + RES_NT - 1) / RES_NT * RES_NT;
  if (per > 65535) return false;                                   // live lists hold 16-bit slice offsets
  if (res_layout((int)per, G, C).bytes > RES_SMEM_BUDGET) return false;
  *SL_out = (int)per;
  return true;
}

// The resident slice as a source of the root find (see "element sources" in prox.cuh).  LC: tax lots and / or per-asset caps.
template <bool LC>
struct SrcRes {
  int C, rank, capw, n_slice, G, Gb;
  int64_t i_beg, row;                      // first asset of the slice; a * N
  double lo_a, hi_a, icg;
  const double *invd, *hi_full, *lot_slope, *lot_width;
  const uint8_t* lot_count;
  double *Ts, *ws;
  uint16_t* live;                          // NW sub-lists of capw entries: warp w lists the live assets it classified
  uint8_t* meta;
  int* lcnt;
  uint32_t* seq;
  double* irc;                             // [NW][RES_IRC]
  double *wpart, *inbox, *ginbox, *gbin;
  double *cPg_, *cRg_;                     // per group: constant buys / sells of the dead assets (whole cluster)
  double cPt, cRt;
  int sstride;                             // 1, or the stride of a SAMPLED root find (prism_settings.sample_until): the passes
  double sscale;                           // visit every sstride-th live entry of a warp's list and scale this CTA's sums

  __device__ __forceinline__ double cP() const { return cPt; }
  __device__ __forceinline__ double cR() const { return cRt; }
  __device__ __forceinline__ double cPg(int g) const { return cPg_[g]; }
  __device__ __forceinline__ double cRg(int g) const { return cRg_[g]; }

  // constants of asset i of the slice; ir = 1 / rho_i
  __device__ __forceinline__ void make(int i, double ir, ElemConst& e, int& g, int& nl, const double*& sl, const double*& wd) const {
    const int64_t gi = i_beg + i;
    e.T = Ts[i]; e.w0 = ws[i];
    e.ir = ir;
    const int m = meta[i];
    g = m & 63;
    double lo = lo_a, hi = hi_a;
    if (LC && hi_full) hi = hi_full[row + gi];
    if (m & 64) { lo = 0.0; hi = 0.0; }
    elem_ranges(e, lo, hi);
    nl = 0; sl = nullptr; wd = nullptr;
    if (LC && lot_count) { nl = lot_count[row + gi]; sl = lot_slope + (row + gi) * PRISM_MAX_LOTS; wd = lot_width + (row + gi) * PRISM_MAX_LOTS; }
  }
  // 1 / rho of entry j of warp wid's sub-list (cached for the first RES_IRC entries, else from global memory)
  __device__ __forceinline__ double ir_of(int wid, int j, int i) const {
    return j < RES_IRC ? irc[wid * RES_IRC + j] : invd[i_beg + i] * icg;
  }
  // live assets of this CTA's slice: warp w walks its own sub-list, the loads of four entries issued together
  template <class F>
  __device__ __forceinline__ void for_each(F f) const {
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint16_t* L = live + wid * capw;
    const int n = lcnt[wid];
    if (sstride > 1) {                       // sampled pass
      for (int j = lane * sstride; j < n; j += 32 * sstride) {
        const int i = L[j];
        ElemConst e; int g, nl; const double *sl, *wd;
        make(i, ir_of(wid, j, i), e, g, nl, sl, wd);
        f(i_beg + i, e, g, nl, sl, wd);
      }
      return;
    }
    int j = lane;
    for (; j + 96 < n; j += 128) {
      int i4[4]; double r4[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) i4[u] = L[j + 32 * u];
#pragma unroll
      for (int u = 0; u < 4; ++u) r4[u] = ir_of(wid, j + 32 * u, i4[u]);
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        ElemConst e; int g, nl; const double *sl, *wd;
        make(i4[u], r4[u], e, g, nl, sl, wd);
        f(i_beg + i4[u], e, g, nl, sl, wd);
      }
    }
    for (; j < n; j += 32) {
      const int i = L[j];
      ElemConst e; int g, nl; const double *sl, *wd;
      make(i, ir_of(wid, j, i), e, g, nl, sl, wd);
      f(i_beg + i, e, g, nl, sl, wd);
    }
  }
  // Reduction over the whole cluster, result identical (bitwise) in every thread of every CTA: warp butterflies, the
  // warp partials added in warp order, the CTA partials sent to every peer's inbox, one cluster barrier, added in
  // rank order.  The inbox is double-buffered (a fast CTA may already be sending the next reduction).
  template <int NV, int OP>
  __device__ __forceinline__ void reduce(double (&val)[NV], double*) const {
    static_assert(NV <= RES_NV, "reduction too wide");
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      double x = val[q];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) x = red_op<OP>(x, __shfl_xor_sync(0xffffffffu, x, o));
      if (lane == 0) wpart[wid * RES_NV + q] = x;
    }
    __syncthreads();
    if (C == 1) {
#pragma unroll
      for (int q = 0; q < NV; ++q) {
        double x = wpart[q];
#pragma unroll
        for (int w = 1; w < RES_NW; ++w) x = red_op<OP>(x, wpart[w * RES_NV + q]);
        val[q] = OP == 0 ? x * sscale : x;
      }
      __syncthreads();
      return;
    }
    const uint32_t buf = seq[tid] & 1u;
    seq[tid] += 1u;
    double* box = inbox + (size_t)buf * C * RES_NV;
    if (tid < NV * C) {
      const int q = tid % NV, r = tid / NV;
      double x = wpart[q];
#pragma unroll
      for (int w = 1; w < RES_NW; ++w) x = red_op<OP>(x, wpart[w * RES_NV + q]);
      res_store_peer(box + rank * RES_NV + q, (uint32_t)r, OP == 0 ? x * sscale : x);
    }
    res_cluster_barrier();
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      double x = box[q];
      for (int r = 1; r < C; ++r) x = red_op<OP>(x, box[r * RES_NV + q]);
      val[q] = x;
    }
  }
  // the per-warp group bins gbin[NW][4 Gb] summed over warps (warp order) and sent to every CTA; afterwards every thread
  // may read the cluster-wide sum of column t with gcol(box, t).  (One cluster barrier; double-buffered like the inbox.)
  template <int NQ>
  __device__ __forceinline__ const double* gather_groups() const {
    const int tid = threadIdx.x;
    const int ncol = NQ * Gb;
    const uint32_t buf = seq[tid] & 1u;
    seq[tid] += 1u;
    double* box = ginbox + (size_t)buf * C * 4 * Gb;
    __syncthreads();
    for (int t = tid; t < ncol; t += RES_NT) {
      double x = gbin[t];
#pragma unroll
      for (int w = 1; w < RES_NW; ++w) x += gbin[w * 4 * Gb + t];
      if (C == 1) box[t] = x;
      else for (int r = 0; r < C; ++r) res_store_peer(box + (size_t)rank * 4 * Gb + t, (uint32_t)r, x);
    }
    if (C == 1) __syncthreads(); else res_cluster_barrier();
    return box;
  }
  __device__ __forceinline__ double gcol(const double* box, int t) const {
    double x = box[t];
    for (int r = 1; r < C; ++r) x += box[(size_t)r * 4 * Gb + t];
    return x;
  }
  // every warp clears its own bins (the previous gather's readers are past a barrier by now)
  __device__ __forceinline__ void zero_bins(int ncol) const {
    double* bins = gbin + (size_t)(threadIdx.x >> 5) * 4 * Gb;
    for (int t = threadIdx.x & 31; t < ncol; t += 32) bins[t] = 0.0;
    __syncwarp();
  }
};

// One pass over the live lists of the cluster: per group g the buys, sells and their slopes at thresholds
// (al + lambda_g, bd + lambda_g)  ->  returned box, column 4 g + {0: P_g, 1: R_g, 2: sP_g, 3: sR_g} (read with gcol).
template <bool LC>
__device__ __noinline__ const double* res_pass_groups(const SrcRes<LC>& s, const double* lamS, double al, double bd) {
  s.zero_bins(4 * s.Gb);
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint16_t* L = s.live + wid * s.capw;
  const int n = s.lcnt[wid];
  double* bins = s.gbin + (size_t)wid * 4 * s.Gb;
  for (int j0 = 0; j0 < n; j0 += 128) {
    int i4[4]; double r4[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int j = j0 + 32 * u + lane; i4[u] = j < n ? L[j] : 0; }
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int j = j0 + 32 * u + lane; r4[u] = j < n ? s.ir_of(wid, j, i4[u]) : 0.0; }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (j0 + 32 * u >= n) break;                       // (warp-uniform)
      const bool valid = j0 + 32 * u + lane < n;
      double x[4] = {0.0, 0.0, 0.0, 0.0};
      int g = 0;
      if (valid) {
        ElemConst e; int nl; const double *sl, *wd;
        s.make(i4[u], r4[u], e, g, nl, sl, wd);
        const double lg = lamS[g];
        x[0] = buy_amt(e, al + lg, x[2]);
        x[1] = sell_amt<LC>(e, bd + lg, sl, wd, nl, x[3]);
      }
      res_group_add<4>(bins, g, x, valid);
    }
  }
  return s.template gather_groups<4>();
}

// the nested robust solver's all-groups pass through the same lean pass
template <bool LC>
__device__ __noinline__ void prox_group_sums(const SrcRes<LC>& s, const double* lamS, int G, double al, double bd,
                                             const double* gw0, double*, double* gsum) {
  const double* box = res_pass_groups<LC>(s, lamS, al, bd);
  for (int g = threadIdx.x; g < G; g += RES_NT)
    gsum[g] = gw0[g] + (s.gcol(box, 4 * g) + s.cPg(g)) - (s.gcol(box, 4 * g + 1) + s.cRg(g));
  __syncthreads();
}

// per-group constants of the dead assets from the warps' bins (columns 2 g + {0, 1}) -> cPg, cRg, totals
template <bool LC>
__device__ __forceinline__ void res_publish_constants(SrcRes<LC>& s) {
  const double* box = s.template gather_groups<2>();
  for (int g = threadIdx.x; g < s.Gb; g += RES_NT) { s.cPg_[g] = s.gcol(box, 2 * g); s.cRg_[g] = s.gcol(box, 2 * g + 1); }
  __syncthreads();
  if (threadIdx.x == 0) {
    double sp = 0.0, sr = 0.0;
    for (int g = 0; g < s.Gb; ++g) { sp += s.cPg_[g]; sr += s.cRg_[g]; }
    s.cPt = sp; s.cRt = sr;
  }
  __syncthreads();
}

// Rare path: every asset of the resident slice live (the solution left the window); only assets that cannot trade at
// all (excluded, lo = hi) stay constants.
template <bool LC>
__device__ __noinline__ void res_reclassify_all(SrcRes<LC>& s) {
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned lt = (1u << lane) - 1u;
  s.zero_bins(2 * s.Gb);
  uint16_t* L = s.live + wid * s.capw;
  double* bins = s.gbin + (size_t)wid * 4 * s.Gb;
  const int nslot = (s.n_slice + RES_NT - 1) / RES_NT;
  int n = 0;
  for (int j = 0; j < nslot; ++j) {
    const int t = j * RES_NT + tid;
    const bool valid = t < s.n_slice;
    bool lv = false;
    double x[2] = {0.0, 0.0};
    int g = 0;
    double ir = 0.0;
    if (valid) {
      ElemConst e; int nl; const double *sl, *wd;
      ir = s.invd[s.i_beg + t] * s.icg;
      s.make(t, ir, e, g, nl, sl, wd);
      lv = e.wB > 0.0 || e.wS > 0.0 || !(e.T == e.T);
      if (!lv) { x[0] = e.bl; x[1] = e.sl; }
    }
    const unsigned m = __ballot_sync(0xffffffffu, lv);
    if (lv) {
      const int pos = n + __popc(m & lt);
      L[pos] = (uint16_t)t;
      if (pos < RES_IRC) s.irc[wid * RES_IRC + pos] = ir;
    }
    n += __popc(m);
    if (__any_sync(0xffffffffu, x[0] != 0.0 || x[1] != 0.0)) res_group_add<2>(bins, g, x, valid && !lv, s.G == 0);
  }
  if (lane == 0) s.lcnt[wid] = n;
  res_publish_constants(s);
}

// Rare path: residual terms (do_check) and / or outputs of EVERY asset of the resident slice at the final thresholds
// (after a window failure or a rho change: the outputs written by the streaming pass are stale).  mx: the seven maxima.
template <bool LC>
__device__ __noinline__ void res_full_pass(const ProxArgs& p, const SrcRes<LC>& s, const double* lamS, int a, double alpha,
                                           double bdf, double lam_b, double gam, double c, double c_new, bool do_check,
                                           bool do_out, bool finished, bool w_out, double* mx) {
  const int tid = threadIdx.x;
  const int64_t row = (int64_t)a * p.N, rowp = (int64_t)a * p.ldw;
  const double cg = c * gam, cgn = c_new * gam, igc = 1.0 / (gam * (1.0 + c_new)), icgn = 1.0 / cgn;
  const bool rescale = c_new != c;
  double nx = 0, nz = 0, nrp = 0, nrd = 0, nPx = 0, ny = 0, nq = 0;
  for (int t = tid; t < s.n_slice; t += RES_NT) {
    const int64_t gi = s.i_beg + t;
    const double iv = p.invd[gi], di = p.d[gi];
    ElemConst e; int g, nl; const double *sl, *wd;
    s.make(t, iv * s.icg, e, g, nl, sl, wd);
    const double lg = lamS[g];
    double mvb, mvs;
    const double tr = buy_amt(e, alpha + lg, mvb) - sell_amt<LC>(e, bdf + lg, sl, wd, nl, mvs);
    const double z = e.w0 + tr;
    const double y = e.T + lam_b - tr * (cg * di);         // rho_old (v - z): unchanged by a rho change
    const double qi = p.q ? p.q[rowp + gi] : -p.mu[row + gi];
    if (do_check) {
      const double x = p.xs[rowp + gi], pq = p.pxq[rowp + gi];
      nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
      nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq - qi)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qi));
      if (!(z == z) || !(x == x) || !(e.T == e.T) || !(pq == pq)) nrp = INFINITY;     // fmax drops NaN: poison explicitly
    }
    if (do_out) {
      if (w_out) p.w_out[row + gi] = z;
      if (!finished) {
        if (rescale) p.v[rowp + gi] = z + y * iv * icgn;   // v' = z + y / rho_new
        const double r = cgn * di * z - y - qi;
        const double rt = r * iv * igc;                    // M_i = gamma d_i (1 + c)
        p.rt[rowp + gi] = rt;
        p.cc[rowp + gi] = rt - z;
      }
    }
  }
  if (do_check) { mx[0] = nx; mx[1] = nz; mx[2] = nrp; mx[3] = nrd; mx[4] = nPx; mx[5] = ny; mx[6] = nq; }
}

// ------------------------------------------------------------------------------------------------ the kernel
// grid = (C, accounts), cluster = (C, 1, 1), block = RES_NT.  mode: PROX_FINAL or 0 (CHECK is the template flag).
template <bool LC, bool CHECK>
__global__ void __launch_bounds__(RES_NT, 2) k_prox_res(const __grid_constant__ ProxArgs p, int mode) {
  extern __shared__ __align__(16) unsigned char res_raw[];
  __shared__ SrcRes<LC> src;
  __shared__ ProxShared sh;
  const int a = blockIdx.y;
  if (p.ap.done[a]) return;                  // (uniform over the cluster)
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int G = p.G, Gb = G > 0 ? G : 1;
  const int C = p.res_C, SL = p.res_SL;
  const int rank = C > 1 ? (int)res_cta_rank() : 0;
  const int64_t N = p.N, row = (int64_t)a * N, rowp = (int64_t)a * p.ldw;
  const int64_t i_beg = (int64_t)rank * SL;
  const int n_slice = (int)max((int64_t)0, min((int64_t)SL, N - i_beg));
  const int nslot = (n_slice + RES_NT - 1) / RES_NT;              // assets per thread (uniform over the CTA)
  const ResLayout lay = res_layout(SL, G, C);
  double* Ts = (double*)(res_raw + lay.Ts);
  double* ws = (double*)(res_raw + lay.ws);
  uint16_t* live = (uint16_t*)(res_raw + lay.live);
  uint8_t* metaS = res_raw + lay.meta;
  int* lcnt = (int*)(res_raw + lay.lcnt);
  double* irc = (double*)(res_raw + lay.irc);
  double* nst = (double*)(res_raw + lay.nst);
  double* grp = (double*)(res_raw + lay.grp);
  double *lamS = grp, *lamW = grp + Gb, *band_lo = grp + 2 * Gb, *band_hi = grp + 3 * Gb, *gw0 = grp + 4 * Gb,
         *gsum = grp + 5 * Gb, *cPg = grp + 6 * Gb, *cRg = grp + 7 * Gb;
  int* act = (int*)(grp + 8 * Gb);
  int* selS = act + 2 * Gb;
  const int capw = SL / RES_NW;
  const bool finalm = (mode & PROX_FINAL) != 0;

  // ---- account constants
  const double gam = p.gamma[a], c = p.ap.c[a], cg = c * gam, icg = 1.0 / cg;
  const double kappa = p.kappa ? p.kappa[a] : 0.0;
  const double lam_b = kappa + (p.c_buy ? p.c_buy[a] : 0.0), Delta = lam_b + kappa;
  const double tau = p.tau ? p.tau[a] : INFINITY;
  const double lo_a = p.lo[a], hi_a = p.hi[a];
  const double b = p.ap.bsum[a];
  const double igc = 1.0 / (gam * (1.0 + c));
  double aw = p.ap.alpha[a], bw = p.ap.beta[a];
  int amode_w = p.ap.mode[a];
  if (!(amode_w == 1 && isfinite(tau))) { amode_w = 0; bw = aw; }
  double W = p.ap.win[a];
  const int nadapt_prev = p.ap.nadapt[a];     // read before anybody writes it
  const bool exact = CHECK || finalm;
  // band ramp: non-check launches of the first iterations project without the group bands (multipliers 0); see DESIGN.md
  const bool bands_on = G > 0 && (exact || p.iter > p.band_start);
  if (G > 0 && !exact && p.iter == p.band_start + 1) W = INFINITY;       // the launch in which the bands join: thresholds jump

  if (tid == 0) {
    src.C = C; src.rank = rank; src.capw = capw; src.n_slice = n_slice; src.G = G; src.Gb = Gb;
    src.i_beg = i_beg; src.row = row; src.lo_a = lo_a; src.hi_a = hi_a; src.icg = icg;
    src.invd = p.invd; src.hi_full = p.hi_full; src.lot_slope = p.lot_slope; src.lot_width = p.lot_width; src.lot_count = p.lot_count;
    src.Ts = Ts; src.ws = ws; src.live = live; src.meta = metaS; src.lcnt = lcnt;
    src.seq = (uint32_t*)(res_raw + lay.seq); src.irc = irc;
    src.wpart = (double*)(res_raw + lay.wpart); src.inbox = (double*)(res_raw + lay.inbox);
    src.ginbox = (double*)(res_raw + lay.ginbox); src.gbin = (double*)(res_raw + lay.gbin);
    src.cPg_ = cPg; src.cRg_ = cRg; src.cPt = 0.0; src.cRt = 0.0; src.sstride = 1; src.sscale = 1.0;
    sh.scratch = nst; sh.gbin = src.gbin; sh.lamS = lamS; sh.gsum = gsum; sh.selS = selS;
    sh.band_lo = band_lo; sh.band_hi = band_hi; sh.gw0 = gw0;
    res_mbar_init((uint64_t*)(res_raw + lay.mbar), 1);
  }
  ((uint32_t*)(res_raw + lay.seq))[tid] = 0u;
  for (int g = tid; g < Gb; g += RES_NT) {
    double l = 0.0;
    if (g < G) {
      const int64_t e = (int64_t)a * G + g;
      band_lo[g] = p.band_lo[e]; band_hi[g] = p.band_hi[e]; gw0[g] = p.gw0[e];
      l = bands_on ? p.lamG[e] : 0.0;
    }
    lamS[g] = l; lamW[g] = l; cPg[g] = 0.0; cRg[g] = 0.0;
  }
  __syncthreads();
  if (C > 1) res_cluster_barrier();          // every CTA of the cluster is running before any peer store

  // ---- A. one pass over the slice (see the header).  v and w0 come by bulk copy (TMA engine) straight into the resident
  // arrays when their rows are 16-byte aligned; the other streams are plain loads, RU assets per thread in flight.
  const unsigned lt = (1u << lane) - 1u;
  const double* vrow = p.v + rowp + i_beg;
  const double* w0row = p.w0 + row + i_beg;
  uint64_t* mbar = (uint64_t*)(res_raw + lay.mbar);
  const int n2 = n_slice & ~1;
  const bool bulk = n2 > 0 && (((uintptr_t)vrow | (uintptr_t)w0row) & 15) == 0;
  if (tid == 0 && bulk) {
    res_mbar_expect(mbar, (uint32_t)n2 * 16u);
    res_bulk_g2s(Ts, vrow, (uint32_t)n2 * 8u, mbar);
    res_bulk_g2s(ws, w0row, (uint32_t)n2 * 8u, mbar);
  }
  double nx = 0, nz = 0, nrp = 0, nrd = 0, nPx = 0, ny = 0, nq = 0;      // residual terms (check launches)
  {
    constexpr int RU = (CHECK || LC) ? 2 : RES_U;
    src.zero_bins(2 * Gb);
    // window in threshold space: a = alpha + lambda_g in [aw + lg - W, aw + lg + W], b - Delta likewise (W = inf: all live)
    const double aN_lo = aw - W, aN_hi = aw + W, bN_lo = bw - W - Delta, bN_hi = bw + W - Delta;
    uint16_t* L = live + wid * capw;
    double* bins = src.gbin + (size_t)wid * 4 * Gb;
    const double* qsrc = p.q ? p.q + rowp + i_beg : p.mu + row + i_beg;
    const double qsgn = p.q ? -1.0 : 1.0;                                 // qm = -q_i
    if (bulk) res_mbar_wait(mbar, 0u);
    int n = 0;
    for (int j0 = 0; j0 < nslot; j0 += RU) {
      double v4[RU], w4[RU], q4[RU], d4[RU], iv4[RU], hi4[RU], s14[RU], x4[RU], pq4[RU];
      int m4[RU], nl4[RU];
#pragma unroll
      for (int u = 0; u < RU; ++u) {
        const int t = (j0 + u) * RES_NT + tid;
        v4[u] = 0.0; w4[u] = 0.0; q4[u] = 0.0; d4[u] = 1.0; iv4[u] = 1.0; hi4[u] = hi_a; s14[u] = 0.0; x4[u] = 0.0; pq4[u] = 0.0;
        m4[u] = 0; nl4[u] = 0;
        if (t < n_slice) {
          const int64_t gi = i_beg + t;
          if (bulk && t < n2) { v4[u] = Ts[t]; w4[u] = ws[t]; } else { v4[u] = vrow[t]; w4[u] = w0row[t]; }
          d4[u] = p.d[gi]; iv4[u] = p.invd[gi];
          if (!finalm) q4[u] = qsrc[t];
          int m = G ? p.group_id[gi] : 0;
          if (p.excl && p.excl[row + gi]) m |= 64;
          m4[u] = m;
          if (LC) {
            if (p.hi_full) hi4[u] = p.hi_full[row + gi];
            if (p.lot_count) { nl4[u] = p.lot_count[row + gi]; s14[u] = p.lot_slope[(row + gi) * PRISM_MAX_LOTS]; }
          }
          if (CHECK && !finalm) { x4[u] = p.xs[rowp + gi]; pq4[u] = p.pxq[rowp + gi]; }
        }
      }
#pragma unroll
      for (int u = 0; u < RU; ++u) {
        if (j0 + u >= nslot) break;                          // (uniform)
        const int t = (j0 + u) * RES_NT + tid;
        const bool valid = t < n_slice;
        const double w0 = w4[u], uu = v4[u] - w0, rho = cg * d4[u];
        const double T = fma(uu, rho, -lam_b);
        const int g = m4[u] & 63;
        const bool ex = (m4[u] & 64) != 0;
        const double tA = T - lamW[g];
        const double hi_i = LC ? hi4[u] : hi_a;
        // Inside its box an asset's buy amount is 0 if the buy threshold of the window cannot reach it, the whole room wB
        // if even the far end of the window fills it, and depends on the thresholds (live) in between; same for sells.
        const bool inbox = w0 >= lo_a && w0 <= hi_i;
        const double wB = hi_i - w0, wS = w0 - lo_a;
        const bool b_reach = tA > aN_lo, b_full = tA - aN_hi >= wB * rho;
        bool s_reach = tA < bN_hi, s_full = bN_lo - tA >= wS * rho;
        if (LC && nl4[u] > 0) { s_reach = tA + s14[u] < bN_hi; s_full = false; }      // lots: no sale anywhere in the window, or live
        double bcst = (b_reach && b_full) ? wB : 0.0, scst = (s_reach && s_full) ? wS : 0.0;
        bool lv = (b_reach && !b_full) || (s_reach && !s_full) || !inbox;             // outside its box (rare): live
        if (ex) { bcst = 0.0; scst = w0; lv = !(w0 >= 0.0); }                          // lo = hi = 0: the trade is -w0
        lv = lv && valid;
        if (valid) {
          Ts[t] = T; metaS[t] = (uint8_t)m4[u];
          if (!(bulk && t < n2)) ws[t] = w0;
        }
        const double tc = bcst - scst, z = w0 + tc;
        if (valid && !lv) {                                  // dead: finished here
          const int64_t gi = i_beg + t;
          if (!finalm) {
            const double rt = fma(rho, (w0 - uu) + 2.0 * tc, qsgn * q4[u]) * (iv4[u] * igc);   // (rho (2 z - v) - q) / M_i
            p.rt[rowp + gi] = rt;
            p.cc[rowp + gi] = rt - z;
          }
          if (CHECK) {
            p.w_out[row + gi] = z;                           // kept if the account finishes here
            if (!finalm) {
              const double x = x4[u], pq = pq4[u], qm = qsgn * q4[u], y = rho * (uu - tc);
              nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
              nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq + qm)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qm));
              if (!(x == x) || !(pq == pq) || !(z == z) || !(T == T)) nrp = INFINITY;
            }
          }
        }
        const unsigned m = __ballot_sync(0xffffffffu, lv);
        if (m) {
          if (lv) {
            const int pos = n + __popc(m & lt);
            L[pos] = (uint16_t)t;
            if (pos < RES_IRC) irc[wid * RES_IRC + pos] = iv4[u] * icg;
          }
          n += __popc(m);
        }
        const bool cst = valid && !lv && (bcst != 0.0 || scst != 0.0);
        if (__any_sync(0xffffffffu, cst)) { const double x2[2] = {bcst, scst}; res_group_add<2>(bins, g, x2, cst, G == 0); }
      }
    }
    if (lane == 0) lcnt[wid] = n;
    res_publish_constants(src);
  }

  // ---- B. root find
  // Sampled root find (prism_settings.sample_until): plain launches of the first iterations, while no band is in the
  // projection, find the thresholds on every stride-th live entry of each warp's list (at most 64 per warp, scaled) and
  // apply them to all live assets: an inexact prox where exactness buys nothing yet.
  const bool sampm = !exact && !bands_on && p.iter < p.sample_until;
  if (sampm) {
    __syncthreads();
    if (tid == 0) {
      int mx = 0;
      for (int w = 0; w < RES_NW; ++w) mx = max(mx, lcnt[w]);
      const int st = (mx + 63) / 64;
      src.sstride = st < 1 ? 1 : st; src.sscale = (double)src.sstride;
    }
    __syncthreads();
  }
  const double tol = 2e-15 * fmax(1.0, fabs(b) + (isfinite(tau) ? tau : 0.0));
  const double Pt = 0.5 * (tau + b), Rt = 0.5 * (tau - b);
  RootState rs;
  rs.n_eval = 0; rs.capped = 0; rs.nobands = bands_on ? 0 : 1;
  double mv = 0.0;
  bool full = false;                         // the window failed: every asset of the slice is re-evaluated below
  for (int att = 0; att < 2; ++att) {
    double al = aw, be = bw;
    int amode = amode_w;
    bool ok = false;
    rs.capped = 0;
    // Newton iteration; where it fails the nested robust solver; where that runs out of Gauss-Seidel rounds over the
    // bands (it converges linearly when several bands interact) the Newton iteration once more from its state, which is
    // close by then (tr = 1); if that fails too, the robust solver from the warm start with as many rounds as it needs
    // (never from the state a failed Newton iteration leaves: see DESIGN.md, readings: robust root find).
    for (int tr = 0; tr < 2; ++tr) {
    ok = false;
    if (!bands_on) {
      // -- plain Newton on P(alpha) = (tau + b)/2, R(beta) = (tau - b)/2 (cap active) or P - R = b (alpha = beta)
      for (int itn = 0; itn < 16; ++itn) {
        double o[12];
        prox_eval<LC>(src, lamS, 0, al, be - Delta, -1, -1, sh.scratch, o);
        ++rs.n_eval;
        const double P = o[0], R = o[1], sP = o[2], sR = o[3];
        const double FA = amode == 1 ? P - Pt : P - R - b, FB = amode == 1 ? R - Rt : 0.0;
        if (fabs(FA) <= tol && fabs(FB) <= tol) {
          if (amode == 1) { if (al >= be) { ok = true; break; } amode = 0; al = be = 0.5 * (al + be); continue; }
          if (!isfinite(tau) || P + R <= tau + tol) { ok = true; break; }
          amode = 1; be = al;
          continue;
        }
        double dal, dbe;
        if (amode == 1) {
          const bool pa_ok = sP > 1e-300, ra_ok = sR > 1e-300;
          if (pa_ok && ra_ok) { dal = FA / sP; dbe = -FB / sR; }
          else if (fabs(FA) <= tol && ra_ok) { dal = 0.0; dbe = -FB / sR; }       // buy side flat and satisfied
          else if (fabs(FB) <= tol && pa_ok) { dbe = 0.0; dal = FA / sP; }        // sell side flat and satisfied
          else break;
        } else {
          const double den = sP + sR;
          if (!(den > 1e-300)) break;
          dal = dbe = FA / den;
        }
        if (!(dal == dal) || !(dbe == dbe)) break;
        al += dal; be += dbe;
      }
    } else {
      // -- semismooth Newton on (alpha, beta, lambda_g of the active bands) jointly, one pass per step: eliminating
      // d lambda_g = (F_g - sP_g d alpha - sR_g d beta) / (sP_g + sR_g) leaves a 2 x 2 system; bands enter the active set
      // when violated and leave it when their multiplier changes sign.  The scalar algebra runs on warp 0 only (lane g
      // owns bands g and g + 32) and is published through shared memory: the other warps just wait at the barrier.
      for (int g = tid; g < G; g += RES_NT) act[g] = lamS[g] > 0.0 ? 1 : (lamS[g] < 0.0 ? -1 : 0);
      __syncthreads();
      for (int itn = 0; itn < 16; ++itn) {
        const double* box = res_pass_groups<LC>(src, lamS, al, be - Delta);
        ++rs.n_eval;
        if (wid == 0) {
          double v13[13];
#pragma unroll
          for (int q = 0; q < 13; ++q) v13[q] = 0.0;
          for (int g = lane; g < G; g += 32) {
            const double Pg = src.gcol(box, 4 * g), Rg = src.gcol(box, 4 * g + 1), pa = src.gcol(box, 4 * g + 2), ra = src.gcol(box, 4 * g + 3);
            const double t = pa + ra;
            const double Sg = gw0[g] + (Pg + cPg[g]) - (Rg + cRg[g]);
            v13[0] += Pg; v13[1] += Rg; v13[2] += pa; v13[3] += ra;
            int ac = act[g];
            if (ac == 0) {
              if (Sg > band_hi[g] + 8.0 * tol) ac = 1; else if (Sg < band_lo[g] - 8.0 * tol) ac = -1;
              if (ac) v13[11] = 1.0;
            }
            if (ac) {
              const double Fg = Sg - (ac > 0 ? band_hi[g] : band_lo[g]);
              if (fabs(Fg) > tol) v13[11] = 1.0;
              if (t > 0.0) { v13[4] += pa * pa / t; v13[5] += ra * ra / t; v13[6] += pa * ra / t; v13[7] += pa * Fg / t; v13[8] += ra * Fg / t; v13[9] += t; v13[10] += Fg; }
              else if (fabs(Fg) > tol) v13[12] = 1.0;
            }
            gsum[g] = Sg;
            act[g] = ac;                                   // (an entering band is active from this step on)
          }
#pragma unroll
          for (int q = 0; q < 13; ++q) v13[q] = warp_sum(v13[q]);
          const double P = src.cPt + v13[0], R = src.cRt + v13[1], sP = v13[2], sR = v13[3];
          const double sA = v13[4], sB = v13[5], sAB = v13[6], rA = v13[7], rB = v13[8], sT = v13[9], sF = v13[10];
          const bool gconv = !(v13[11] > 0.0), sing = v13[12] > 0.0;
          const double FA = amode == 1 ? P - Pt : P - R - b, FB = amode == 1 ? R - Rt : 0.0;
          int code = 0;                                    // 0: step taken, 1: converged, 2: give up (robust solver)
          double dal = 0.0, dbe = 0.0;
          bool step = false;
          if (fabs(FA) <= tol && fabs(FB) <= tol && gconv) {
            if (amode == 1) { if (al >= be) code = 1; else { amode = 0; al = be = 0.5 * (al + be); } }
            else if (!isfinite(tau) || P + R <= tau + tol) code = 1;
            else { amode = 1; be = al; }
          } else if (sing) code = 2;
          else {
            step = true;
            if (amode == 1) {
              const double M11 = -sP + sA, M12 = sAB, M21 = -sAB, M22 = sR - sB, r1 = -FA + rA, r2 = -FB - rB;
              const double det = M11 * M22 - M12 * M21;
              if (fabs(det) > 1e-300) { dal = (r1 * M22 - M12 * r2) / det; dbe = (M11 * r2 - M21 * r1) / det; }
              else if (fabs(r1) <= tol && fabs(M11) <= 1e-300 && fabs(M22) > 1e-300) { dal = 0.0; dbe = r2 / M22; }
              else if (fabs(r2) <= tol && fabs(M22) <= 1e-300 && fabs(M11) > 1e-300) { dbe = 0.0; dal = r1 / M11; }
              else code = 2;
            } else {
              const double den = (sP + sR) - sT;
              if (!(den > 1e-300)) code = 2; else dal = dbe = (FA - sF) / den;
            }
            if (!(dal == dal) || !(dbe == dbe)) code = 2;
          }
          if (step && code == 0) {
            for (int g = lane; g < G; g += 32) {           // multipliers and active set
              const double pa = src.gcol(box, 4 * g + 2), ra = src.gcol(box, 4 * g + 3), t = pa + ra;
              int ac = act[g];
              if (ac && t > 0.0) {
                const double Fg = gsum[g] - (ac > 0 ? band_hi[g] : band_lo[g]);
                double ln = lamS[g] + (Fg - pa * dal - ra * dbe) / t;
                if (!(ln * ac > 0.0)) { ln = 0.0; ac = 0; } // the multiplier would change sign: the band goes inactive
                lamS[g] = ln;
              }
              act[g] = ac;
            }
            al += dal; be += dbe;
          }
          if (lane == 0) { nst[0] = al; nst[1] = be; nst[2] = (double)amode; nst[3] = (double)code; }
        }
        __syncthreads();
        al = nst[0]; be = nst[1]; amode = (int)nst[2];
        const int code = (int)nst[3];
        __syncthreads();                                   // nst is rewritten by the next step
        if (code == 1) { ok = true; break; }
        if (code == 2) break;
      }
    }
    if (ok) { rs.alpha = al; rs.beta = be; rs.amode = amode; rs.capped = 0; break; }
    {
      // nested robust solver (prox.cuh) on the same live lists; continues from the Newton state when that is usable
      // (not with an infinite window while bands are in play: see DESIGN.md, readings: robust root find)
      const bool keep = tr > 0 ? false
                               : (al == al && be == be && fabs(al - aw) <= 0.5 * W && fabs(be - bw) <= 0.5 * W && (W < INFINITY || !bands_on));
      __syncthreads();
      if (!keep) for (int g = tid; g < G; g += RES_NT) lamS[g] = lamW[g];
      __syncthreads();
      rs.alpha = keep ? al : aw; rs.beta = keep ? be : bw; rs.amode = keep ? amode : amode_w;
      rs.max_rounds = (bands_on && tr < 1) ? 2 * G + 2 : (1 << 30);
      prox_rootfind<LC>(p, src, a, b, tau, Delta, sh, rs);
      if (rs.capped != 2) break;
      al = rs.alpha; be = rs.beta; amode = rs.amode;
    }
    }
    double mv_l = 0.0;
    if (bands_on) for (int g = 0; g < G; ++g) mv_l = fmax(mv_l, fabs(lamS[g] - lamW[g]));
    mv = fmax(fmax(fabs(rs.alpha - aw), fabs(rs.beta - bw)), mv_l);
    if (sampm || !(W < INFINITY) || mv <= 0.5 * W) break;   // (a sampled solve is inexact by design: no reclassification)
    // the solution left the window the live lists were built for: every asset live, solve again from the warm start
    __syncthreads();
    for (int g = tid; g < G; g += RES_NT) lamS[g] = lamW[g];
    W = INFINITY;
    full = true;
    res_reclassify_all(src);
  }
  __syncthreads();
  const double alpha = rs.alpha, beta = rs.beta, bdf = beta - Delta;

  // outputs (and residual terms) of the live assets of this warp's sub-list
  auto live_pass = [&](bool do_check, bool do_out, bool finished) {
    const uint16_t* L = live + wid * capw;
    const int n = lcnt[wid];
    for (int j = lane; j < n; j += 32) {
      const int t = L[j];
      const int64_t gi = i_beg + t;
      const double iv = p.invd[gi], di = p.d[gi];
      const double qi = p.q ? p.q[rowp + gi] : -p.mu[row + gi];
      double x = 0.0, pq = 0.0;
      if (do_check) { x = p.xs[rowp + gi]; pq = p.pxq[rowp + gi]; }
      ElemConst e; int g, nl; const double *sl, *wd;
      src.make(t, iv * icg, e, g, nl, sl, wd);
      const double lg = lamS[g];
      double mvb, mvs;
      const double tr = buy_amt(e, alpha + lg, mvb) - sell_amt<LC>(e, bdf + lg, sl, wd, nl, mvs);
      const double z = e.w0 + tr;
      const double y = e.T + lam_b - tr * (cg * di);
      if (do_check) {
        nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
        nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq - qi)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qi));
        if (!(z == z) || !(x == x) || !(e.T == e.T) || !(pq == pq)) nrp = INFINITY;
      }
      if (do_out) {
        if (CHECK) p.w_out[row + gi] = z;
        if (!finished) {
          const double r = cg * di * z - y - qi;
          const double rt = r * iv * igc;
          p.rt[rowp + gi] = rt;
          p.cc[rowp + gi] = rt - z;
        }
      }
    }
  };

  // ---- check: scaled residuals of the splitting (reading R13), convergence mask (H6), rho adaptation (H7)
  double c_new = c;
  int finished = 0;
  if (CHECK && !finalm) {
    if (full) {                              // the terms gathered by the streaming pass assumed the window held
      double mx[7];
      res_full_pass<LC>(p, src, lamS, a, alpha, bdf, lam_b, gam, c, c, true, false, false, false, mx);
      nx = mx[0]; nz = mx[1]; nrp = mx[2]; nrd = mx[3]; nPx = mx[4]; ny = mx[5]; nq = mx[6];
    } else live_pass(true, false, false);
    double val[7] = {nx, nz, nrp, nrd, nPx, ny, nq};
    src.template reduce<7, 1>(val, nullptr);
    const double rp = val[2] / fmax(fmax(val[0], val[1]), 1e-300);
    const double rd = val[3] / fmax(fmax(val[4], fmax(val[5], val[6])), 1e-300);
    const bool bad = !(rp < INFINITY) || !(rd < INFINITY) || !(alpha == alpha) || !(beta == beta);
    const bool conv = !bad && val[2] <= p.eps_abs + p.eps * fmax(val[0], val[1]) &&
                      val[3] <= p.eps_abs + p.eps * fmax(val[4], fmax(val[5], val[6])) && !rs.capped;   // never certify on an unfinished root find
    if (tid == 0 && rank == 0) {
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_PRIMAL] = rp;
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_DUAL] = rd;
    }
    if (conv || bad) {
      finished = 1;
      if (tid == 0 && rank == 0) p.ap.conv[a] = bad ? -1 : 1;
    } else if (p.adapt && p.iter >= p.adapt_start && p.iter - nadapt_prev >= p.adapt_every) {
      const double ratio = sqrt(rp / fmax(rd, 1e-300));
      if (ratio > 3.0 || ratio < 1.0 / 3.0) {
        c_new = c * fmin(fmax(ratio, 0.2), 5.0);
        if (tid == 0 && rank == 0) { p.ap.c[a] = c_new; p.ap.refactor[a] = 1; }
      }
      if (tid == 0 && rank == 0) p.ap.nadapt[a] = p.iter;
    }
  }
  if (finalm) finished = 1;

  // ---- C. outputs: the live assets; every asset of the slice after a window failure or a rho change
  if (full || c_new != c) res_full_pass<LC>(p, src, lamS, a, alpha, bdf, lam_b, gam, c, c_new, false, true, finished != 0, CHECK, nullptr);
  else live_pass(false, true, finished != 0);

  // ---- commit the account's state
  if (rank == 0) {
    if (bands_on) for (int g = tid; g < G; g += RES_NT) p.lamG[(int64_t)a * G + g] = lamS[g];
    if (tid == 0) {
      p.ap.alpha[a] = alpha; p.ap.beta[a] = beta; p.ap.mode[a] = rs.amode;
      p.ap.win[a] = next_window(p, alpha, beta, mv);       // next window: a multiple of how far the thresholds moved
      if (finished) {
        p.ap.done[a] = 1;
        p.ap.iters[a] = p.iter;
        atomicAdd(&p.counters[0], 1);
        double* du = p.duals + (int64_t)a * PRISM_NDUAL(G);
        du[0] = 0.5 * (alpha + beta);
        du[1] = 0.5 * (alpha - beta);
        for (int g = 0; g < G; ++g) { du[2 + g] = fmax(lamS[g], 0.0); du[2 + G + g] = fmax(-lamS[g], 0.0); }
        p.resid[(int64_t)a * PRISM_NRES + PRISM_R_RHO] = c_new;
      }
    }
  }
  if (C > 1) res_cluster_barrier();          // no CTA exits while a peer may still address its shared memory
}
