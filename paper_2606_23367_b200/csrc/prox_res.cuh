// prox_res.cuh - the cluster-resident form of the fused proximal / projection step: ONE kernel
// per iteration, one thread-block CLUSTER per account.
//
// The account's assets are cut into C contiguous slices, one per CTA of the cluster (C = 1, 2, 4, 8 or 16, the smallest
// for which a slice fits the shared-memory budget).  Each CTA
//   A. streams its slice once (v, w0, exclusion mask; d, 1/d, group id of the shared universe) and keeps
//      T_i = rho_i (v_i - w0_i) - (kappa + c_buy) and w0_i RESIDENT in shared memory (20 bytes per asset), classifying
//      every asset against the window around the warm-start thresholds on the way: "dead" assets (buy and sell amounts
//      constant for every threshold inside the window) only contribute constants, the others go to a live list;
//   B. takes part in the root find for (alpha, beta, lambda_g) of prox.cuh: every trial evaluation is a pass over the
//      live lists of all C slices out of shared memory, the partial sums meet through DISTRIBUTED shared memory
//      (st.shared::cluster into every peer's inbox + one cluster barrier) and are added in rank order, so every CTA
//      holds bit-identical sums and runs the identical (redundant) scalar logic: a joint semismooth Newton iteration,
//      with the nested bracketed solver prox_rootfind as the robust fallback;
//   C. writes r~ = M^-1 r and c = r~ - z for its slice from the resident T, w0 and the final thresholds (every asset is
//      evaluated with the final thresholds, so the window only ever affects the cost of B, never the result), and on
//      check launches the residual terms, the convergence mask, the rho adaptation and the returned weights.
// Compared with the streaming pair k_prox_stream + k_prox_root (prox_fast.cuh) there are no live lists in global
// memory, no sort, no fixed-point bins, no second launch and no every-asset fallback: a solution that leaves the
// window rebuilds the live list from shared memory and repeats B.  All sums are fp64 in a fixed order (deterministic).
// Tax lots and per-asset caps are handled by the same kernel (template LOTS): lot rows are read from global memory for
// live assets only.
#pragma once
#include "prox.cuh"

#define RES_NT 256                 // threads per CTA (two CTAs per SM at <= 128 registers)
#define RES_NW (RES_NT / 32)
#define RES_NV 16                  // widest cluster-wide reduction (values per call)
#define RES_SMEM_BUDGET (110 * 1024)   // dynamic shared memory per CTA: two CTAs per SM

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

// lanes holding the same group are summed in ascending lane order, the lowest lane adds the sums to this warp's bins
// bins[NQ * g + q] (deterministic; call from warp-uniform control flow)
template <int NQ>
__device__ __forceinline__ void res_group_add(double* bins, int g, const double (&x)[NQ], bool valid) {
  const int lane = threadIdx.x & 31;
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
  size_t Ts, ws, live, gid, cls, lcnt, seq, wpart, inbox, ginbox, gbin, grp, scratch, bytes;
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
  L.grp = o; o += (size_t)10 * Gb * 8;                    // lamS lamW band_lo band_hi gw0 gsum cPg cRg + act, sel (ints)
  L.scratch = o; o += (size_t)12 * 32 * 8;                // work area of prox_rootfind (unused by the cluster reductions)
  L.seq = o; o += (size_t)RES_NT * 4;                     // per-thread reduction counters (inbox parity)
  L.lcnt = o; o += (size_t)RES_NW * 4 + 16;
  L.live = o; o += (size_t)SL * 2;
  L.gid = o; o += (size_t)SL;
  L.cls = o; o += (size_t)SL;
  L.bytes = (o + 15) & ~(size_t)15;
  return L;
}

// The resident slice as a source of the root find (see "element sources" in prox.cuh).
template <bool LOTS>
struct SrcRes {
  int C, rank, capw, n_slice, G, Gb;
  int64_t i_beg, row;                      // first asset of the slice; a * N
  double lo_a, hi_a, icg;
  const double *invd, *hi_full, *lot_slope, *lot_width;
  const uint8_t* lot_count;
  double *Ts, *ws;
  uint16_t* live;                          // NW sub-lists of capw entries: warp w lists the live assets it classified
  uint8_t *gid, *cls;                      // cls bit 0: excluded (lo = hi = 0)
  int* lcnt;
  uint32_t* seq;
  double *wpart, *inbox, *ginbox, *gbin;
  double *cPg_, *cRg_;                     // per group: constant buys / sells of the dead assets (whole cluster)
  double cPt, cRt;

  __device__ __forceinline__ double cP() const { return cPt; }
  __device__ __forceinline__ double cR() const { return cRt; }
  __device__ __forceinline__ double cPg(int g) const { return cPg_[g]; }
  __device__ __forceinline__ double cRg(int g) const { return cRg_[g]; }

  __device__ __forceinline__ void load(int i, ElemConst& e, int& g, int& nl, const double*& sl, const double*& wd) const {
    const int64_t gi = i_beg + i;
    e.T = Ts[i]; e.w0 = ws[i];
    e.ir = invd[gi] * icg;
    g = gid[i];
    double lo = lo_a, hi = hi_full ? hi_full[row + gi] : hi_a;
    if (cls[i] & 1) { lo = 0.0; hi = 0.0; }
    elem_ranges(e, lo, hi);
    nl = 0; sl = nullptr; wd = nullptr;
    if (LOTS) { nl = lot_count[row + gi]; sl = lot_slope + (row + gi) * PRISM_MAX_LOTS; wd = lot_width + (row + gi) * PRISM_MAX_LOTS; }
  }
  // live assets of this CTA's slice: warp w walks its own sub-list
  template <class F>
  __device__ __forceinline__ void for_each(F f) const {
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint16_t* L = live + wid * capw;
    const int n = lcnt[wid];
    for (int j = lane; j < n; j += 32) {
      const int i = L[j];
      ElemConst e; int g, nl; const double *sl, *wd;
      load(i, e, g, nl, sl, wd);
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
        val[q] = x;
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
      res_store_peer(box + rank * RES_NV + q, (uint32_t)r, x);
    }
    res_cluster_barrier();
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      double x = box[q];
      for (int r = 1; r < C; ++r) x = red_op<OP>(x, box[r * RES_NV + q]);
      val[q] = x;
    }
  }
  // the per-warp group bins gbin[NW][NQ Gb] summed over warps (warp order) and CTAs (rank order); afterwards every thread
  // may read the cluster-wide sum of column t with gcol(t).  (One cluster barrier; double-buffered like the inbox.)
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
  __device__ __forceinline__ void zero_bins(int ncol_per_warp_stride_4Gb) const {
    for (int t = threadIdx.x; t < RES_NW * 4 * Gb; t += RES_NT) gbin[t] = 0.0;
    (void)ncol_per_warp_stride_4Gb;
    __syncthreads();
  }
};

// One pass over the live lists of the cluster: per group g the buys, sells and their slopes at thresholds
// (al + lambda_g, bd + lambda_g)  ->  returned box, column 4 g + {0: P_g, 1: R_g, 2: sP_g, 3: sR_g} (read with gcol).
template <bool LOTS>
__device__ __noinline__ const double* res_pass_groups(const SrcRes<LOTS>& s, const double* lamS, double al, double bd) {
  s.zero_bins(0);
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint16_t* L = s.live + wid * s.capw;
  const int n = s.lcnt[wid];
  double* bins = s.gbin + (size_t)wid * 4 * s.Gb;
  for (int j0 = 0; j0 < n; j0 += 32) {
    const int j = j0 + lane;
    const bool valid = j < n;
    double x[4] = {0.0, 0.0, 0.0, 0.0};
    int g = 0;
    if (valid) {
      ElemConst e; int nl; const double *sl, *wd;
      s.load(L[j], e, g, nl, sl, wd);
      const double lg = lamS[g];
      x[0] = buy_amt(e, al + lg, x[2]);
      x[1] = sell_amt<LOTS>(e, bd + lg, sl, wd, nl, x[3]);
    }
    res_group_add<4>(bins, g, x, valid);
  }
  return s.template gather_groups<4>();
}

// the nested robust solver's all-groups pass through the same lean pass
template <bool LOTS>
__device__ __noinline__ void prox_group_sums(const SrcRes<LOTS>& s, const double* lamS, int G, double al, double bd,
                                             const double* gw0, double*, double* gsum) {
  const double* box = res_pass_groups<LOTS>(s, lamS, al, bd);
  for (int g = threadIdx.x; g < G; g += RES_NT)
    gsum[g] = gw0[g] + (s.gcol(box, 4 * g) + s.cPg(g)) - (s.gcol(box, 4 * g + 1) + s.cRg(g));
  __syncthreads();
}

__host__ __device__ inline bool res_fits(int64_t N, int G, int C, int* SL_out) {
  int64_t per = (N + C - 1) / C;
  per = (per + RES_NT - 1) / RES_NT * RES_NT;
  if (per > 65535) return false;                                   // live lists hold 16-bit slice offsets
  if (res_layout((int)per, G, C).bytes > RES_SMEM_BUDGET) return false;
  *SL_out = (int)per;
  return true;
}

// ------------------------------------------------------------------------------------------------ the kernel
// grid = (C, accounts), cluster = (C, 1, 1), block = RES_NT.  mode: PROX_FINAL or 0 (CHECK is the template flag).
template <bool LOTS, bool CHECK>
__global__ void __launch_bounds__(RES_NT, 2) k_prox_res(const __grid_constant__ ProxArgs p, int mode) {
  extern __shared__ __align__(16) unsigned char res_raw[];
  __shared__ SrcRes<LOTS> src;
  __shared__ ProxShared sh;
  __shared__ double bc[2][RES_NV];           // CTA-local broadcast of the joint Newton's reduced terms
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
  uint8_t* gidS = res_raw + lay.gid;
  uint8_t* clsS = res_raw + lay.cls;
  int* lcnt = (int*)(res_raw + lay.lcnt);
  double* grp = (double*)(res_raw + lay.grp);
  double *lamS = grp, *lamW = grp + Gb, *band_lo = grp + 2 * Gb, *band_hi = grp + 3 * Gb, *gw0 = grp + 4 * Gb,
         *gsum = grp + 5 * Gb, *cPg = grp + 6 * Gb, *cRg = grp + 7 * Gb;
  int* act = (int*)(grp + 8 * Gb);
  int* selS = (int*)(grp + 9 * Gb);
  const int capw = SL / RES_NW;

  // ---- account constants
  const double gam = p.gamma[a], c = p.ap.c[a], cg = c * gam, icg = 1.0 / cg;
  const double kappa = p.kappa ? p.kappa[a] : 0.0;
  const double lam_b = kappa + (p.c_buy ? p.c_buy[a] : 0.0), Delta = lam_b + kappa;
  const double tau = p.tau ? p.tau[a] : INFINITY;
  const double lo_a = p.lo[a], hi_a = p.hi[a];
  const double b = p.ap.bsum[a];
  double aw = p.ap.alpha[a], bw = p.ap.beta[a];
  int amode_w = p.ap.mode[a];
  if (!(amode_w == 1 && isfinite(tau))) { amode_w = 0; bw = aw; }
  double W = p.ap.win[a];
  const int nadapt_prev = p.ap.nadapt[a];     // read before anybody writes it
  const bool exact = CHECK || (mode & PROX_FINAL);
  // band ramp: non-check launches of the first iterations project without the group bands (multipliers 0); see DESIGN.md
  const bool bands_on = G > 0 && (exact || p.iter > p.band_start);
  if (G > 0 && !exact && p.iter == p.band_start + 1) W = INFINITY;       // the launch in which the bands join: thresholds jump

  if (tid == 0) {
    src.C = C; src.rank = rank; src.capw = capw; src.n_slice = n_slice; src.G = G; src.Gb = Gb;
    src.i_beg = i_beg; src.row = row; src.lo_a = lo_a; src.hi_a = hi_a; src.icg = icg;
    src.invd = p.invd; src.hi_full = p.hi_full; src.lot_slope = p.lot_slope; src.lot_width = p.lot_width; src.lot_count = p.lot_count;
    src.Ts = Ts; src.ws = ws; src.live = live; src.gid = gidS; src.cls = clsS; src.lcnt = lcnt;
    src.seq = (uint32_t*)(res_raw + lay.seq);
    src.wpart = (double*)(res_raw + lay.wpart); src.inbox = (double*)(res_raw + lay.inbox);
    src.ginbox = (double*)(res_raw + lay.ginbox); src.gbin = (double*)(res_raw + lay.gbin);
    src.cPg_ = cPg; src.cRg_ = cRg; src.cPt = 0.0; src.cRt = 0.0;
    sh.scratch = (double*)(res_raw + lay.scratch); sh.gbin = src.gbin; sh.lamS = lamS; sh.gsum = gsum; sh.selS = selS;
    sh.band_lo = band_lo; sh.band_hi = band_hi; sh.gw0 = gw0;
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

  // ---- A. stream the slice in: T, w0, group, class resident; classify against the window; constants of the dead
  // assets per group.  Window W around (aw, bw, lamW): thresholds a = alpha + lambda_g in [aw + lg - W, aw + lg + W].
  const unsigned lt = (1u << lane) - 1u;
  const double* vrow = p.v + rowp + i_beg;
  const double* w0row = p.w0 + row + i_beg;
  auto classify = [&](bool from_global) {
    // from_global: first classification, fused with the load; else rebuild from the resident slice with W as set
    src.zero_bins(0);
    const bool allw = !(W < INFINITY);
    uint16_t* L = live + wid * capw;
    double* bins = src.gbin + (size_t)wid * 4 * Gb;
    int n = 0;
    for (int j = 0; j < nslot; ++j) {
      const int t = j * RES_NT + tid;
      const bool valid = t < n_slice;
      bool lv = false;
      double x[2] = {0.0, 0.0};
      int g = 0;
      if (valid) {
        const int64_t gi = i_beg + t;
        double T, w0;
        int ex;
        const double iv = p.invd[gi];
        if (from_global) {
          const double v = vrow[t];
          w0 = w0row[t];
          ex = p.excl ? (p.excl[row + gi] != 0) : 0;
          g = G ? p.group_id[gi] : 0;
          T = fma(v - w0, cg * p.d[gi], -lam_b);
          Ts[t] = T; ws[t] = w0; gidS[t] = (uint8_t)g; clsS[t] = (uint8_t)ex;
        } else {
          T = Ts[t]; w0 = ws[t]; g = gidS[t]; ex = clsS[t] & 1;
        }
        ElemConst e;
        e.T = T; e.w0 = w0; e.ir = iv * icg;
        double lo = lo_a, hi = p.hi_full ? p.hi_full[row + gi] : hi_a;
        if (ex) { lo = 0.0; hi = 0.0; }
        elem_ranges(e, lo, hi);
        const double lg = lamW[g];
        // buy side: amount = bl + clamp((T - a) ir - bl, 0, wB), largest at the low end of the window
        bool blive = false, slive = false;
        if (e.wB > 0.0) {
          if (allw) blive = true;
          else {
            const double tmax = (T - (aw + lg - W)) * e.ir - e.bl, tmin = (T - (aw + lg + W)) * e.ir - e.bl;
            if (tmax <= 0.0) {}
            else if (tmin >= e.wB) x[0] += e.wB;
            else blive = true;
          }
        }
        x[0] += e.bl;
        // sell side: amount = sl + clamp((b - Delta - T) ir - sl, 0, wS), largest at the high end of the window
        int nl = 0;
        if (LOTS) nl = p.lot_count[row + gi];
        if (LOTS && nl > 0) {
          // lots: unreachable (no sale anywhere in the window) is the only dead state; forced sales stay live
          const double s1 = p.lot_slope[(row + gi) * PRISM_MAX_LOTS];
          if (allw || e.sl > 0.0 || (bw + lg + W - Delta - s1 - T) > 0.0) slive = true;
        } else if (e.wS > 0.0) {
          if (allw) slive = true;
          else {
            const double tmax = ((bw + lg + W - Delta) - T) * e.ir - e.sl, tmin = ((bw + lg - W - Delta) - T) * e.ir - e.sl;
            if (tmax <= 0.0) {}
            else if (tmin >= e.wS) x[1] += e.wS;
            else slive = true;
          }
          x[1] += e.sl;
        } else x[1] += e.sl;
        lv = blive || slive;
        if (!(T == T)) lv = true;                          // NaN: keep it in the list, the sums turn NaN and the check flags it
        if (lv) { x[0] = 0.0; x[1] = 0.0; }
      }
      const unsigned m = __ballot_sync(0xffffffffu, lv);
      if (lv) L[n + __popc(m & lt)] = (uint16_t)t;
      n += __popc(m);
      if (__any_sync(0xffffffffu, x[0] != 0.0 || x[1] != 0.0)) res_group_add<2>(bins, g, x, valid && !lv);
    }
    if (lane == 0) lcnt[wid] = n;
    // constants: res_group_add<2> wrote columns 2 g + {0, 1} of the warp's bins; gather as 2 Gb columns
    const double* box = src.template gather_groups<2>();
    for (int g = tid; g < Gb; g += RES_NT) { cPg[g] = src.gcol(box, 2 * g); cRg[g] = src.gcol(box, 2 * g + 1); }
    __syncthreads();
    if (tid == 0) {
      double sp = 0.0, sr = 0.0;
      for (int g = 0; g < Gb; ++g) { sp += cPg[g]; sr += cRg[g]; }
      src.cPt = sp; src.cRt = sr;
    }
    __syncthreads();
  };
  classify(true);

  // ---- B. root find
  const double tol = 2e-15 * fmax(1.0, fabs(b) + (isfinite(tau) ? tau : 0.0));
  const double Pt = 0.5 * (tau + b), Rt = 0.5 * (tau - b);
  RootState rs;
  rs.n_eval = 0; rs.capped = 0; rs.nobands = bands_on ? 0 : 1;
  double mv = 0.0;
  for (int att = 0; att < 2; ++att) {
    double al = aw, be = bw;
    int amode = amode_w;
    bool ok = false;
    rs.capped = 0;
    if (!bands_on) {
      // -- plain Newton on P(alpha) = (tau + b)/2, R(beta) = (tau - b)/2 (cap active) or P - R = b (alpha = beta)
      for (int itn = 0; itn < 16; ++itn) {
        double o[12];
        prox_eval<LOTS>(src, lamS, 0, al, be - Delta, -1, -1, sh.scratch, o);
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
      // when violated and leave it when their multiplier changes sign (see k_prox_root in prox_fast.cuh for the algebra)
      for (int g = tid; g < G; g += RES_NT) act[g] = lamS[g] > 0.0 ? 1 : (lamS[g] < 0.0 ? -1 : 0);
      __syncthreads();
      for (int itn = 0; itn < 16; ++itn) {
        const double* box = res_pass_groups<LOTS>(src, lamS, al, be - Delta);
        ++rs.n_eval;
        double v16[RES_NV];
#pragma unroll
        for (int q = 0; q < RES_NV; ++q) v16[q] = 0.0;
        if (tid < 64) {
          for (int g = tid; g < G; g += 64) {
            const double Pg = src.gcol(box, 4 * g), Rg = src.gcol(box, 4 * g + 1), pa = src.gcol(box, 4 * g + 2), ra = src.gcol(box, 4 * g + 3);
            const double t = pa + ra;
            const double Sg = gw0[g] + (Pg + cPg[g]) - (Rg + cRg[g]);
            v16[0] += Pg; v16[1] += Rg; v16[2] += pa; v16[3] += ra;
            int ac = act[g];
            if (ac == 0) {
              if (Sg > band_hi[g] + 8.0 * tol) ac = 1; else if (Sg < band_lo[g] - 8.0 * tol) ac = -1;
              if (ac) v16[11] = 1.0;
            }
            if (ac) {
              const double Fg = Sg - (ac > 0 ? band_hi[g] : band_lo[g]);
              if (fabs(Fg) > tol) v16[11] = 1.0;
              if (t > 0.0) { v16[4] += pa * pa / t; v16[5] += ra * ra / t; v16[6] += pa * ra / t; v16[7] += pa * Fg / t; v16[8] += ra * Fg / t; v16[9] += t; v16[10] += Fg; }
              else if (fabs(Fg) > tol) v16[12] = 1.0;
            }
            gsum[g] = Sg;
          }
#pragma unroll
          for (int q = 0; q < 13; ++q) {
            const double x = warp_sum(v16[q]);
            if (lane == 0) bc[wid][q] = x;
          }
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 13; ++q) v16[q] = bc[0][q] + bc[1][q];
        const double P = src.cPt + v16[0], R = src.cRt + v16[1], sP = v16[2], sR = v16[3];
        const double sA = v16[4], sB = v16[5], sAB = v16[6], rA = v16[7], rB = v16[8], sT = v16[9], sF = v16[10];
        const bool gconv = !(v16[11] > 0.0), sing = v16[12] > 0.0;
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
          else if (fabs(r1) <= tol && fabs(M11) <= 1e-300 && fabs(M22) > 1e-300) { dal = 0.0; dbe = r2 / M22; }
          else if (fabs(r2) <= tol && fabs(M22) <= 1e-300 && fabs(M11) > 1e-300) { dbe = 0.0; dal = r1 / M11; }
          else break;
        } else {
          const double den = (sP + sR) - sT;
          if (!(den > 1e-300)) break;
          dal = dbe = (FA - sF) / den;
        }
        if (!(dal == dal) || !(dbe == dbe)) break;
        for (int g = tid; g < G; g += RES_NT) {            // multipliers and active set (thread g owns band g)
          const double pa = src.gcol(box, 4 * g + 2), ra = src.gcol(box, 4 * g + 3), t = pa + ra;
          int ac = act[g];
          if (ac == 0) { if (gsum[g] > band_hi[g] + 8.0 * tol) ac = 1; else if (gsum[g] < band_lo[g] - 8.0 * tol) ac = -1; }
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
    }
    if (ok) { rs.alpha = al; rs.beta = be; rs.amode = amode; }
    else {
      // nested robust solver (prox.cuh) on the same live lists; continues from the Newton state when that is usable
      // (not with an infinite window while bands are in play: see DESIGN.md, readings: robust root find)
      const bool keep = al == al && be == be && fabs(al - aw) <= 0.5 * W && fabs(be - bw) <= 0.5 * W && (W < INFINITY || !bands_on);
      __syncthreads();
      if (!keep) for (int g = tid; g < G; g += RES_NT) lamS[g] = lamW[g];
      __syncthreads();
      rs.alpha = keep ? al : aw; rs.beta = keep ? be : bw; rs.amode = keep ? amode : amode_w;
      prox_rootfind<LOTS>(p, src, a, b, tau, Delta, sh, rs);
    }
    double mv_l = 0.0;
    for (int g = 0; g < G; ++g) mv_l = fmax(mv_l, fabs(lamS[g] - lamW[g]));
    mv = fmax(fmax(fabs(rs.alpha - aw), fabs(rs.beta - bw)), mv_l);
    if (!(W < INFINITY) || mv <= 0.5 * W) break;
    // the solution left the window the live lists were built for: every asset live, solve again from the warm start
    __syncthreads();
    for (int g = tid; g < G; g += RES_NT) lamS[g] = lamW[g];
    W = INFINITY;
    classify(false);
  }
  __syncthreads();
  const double alpha = rs.alpha, beta = rs.beta, bdf = beta - Delta;

  // trade of asset t of the slice at the final thresholds
  auto trade = [&](int t, int64_t gi, double T, double w0, double iv) -> double {
    ElemConst e;
    e.T = T; e.w0 = w0; e.ir = iv * icg;
    double lo = lo_a, hi = p.hi_full ? p.hi_full[row + gi] : hi_a;
    if (clsS[t] & 1) { lo = 0.0; hi = 0.0; }
    elem_ranges(e, lo, hi);
    const double lg = lamS[gidS[t]];
    double mvb, mvs;
    int nl = 0; const double *sl = nullptr, *wd = nullptr;
    if (LOTS) {
      nl = p.lot_count[row + gi];
      if (nl > 0 && !((bdf + lg - T) > 0.0 || e.sl > 0.0)) nl = -1;       // no sale possible: skip the lot rows
      if (nl > 0) { sl = p.lot_slope + (row + gi) * PRISM_MAX_LOTS; wd = p.lot_width + (row + gi) * PRISM_MAX_LOTS; }
    }
    const double sell = nl < 0 ? 0.0 : sell_amt<LOTS>(e, bdf + lg, sl, wd, nl, mvs);
    return buy_amt(e, alpha + lg, mvb) - sell;
  };

  // ---- check: scaled residuals of the splitting (reading R13), convergence mask (H6), rho adaptation (H7)
  double c_new = c;
  int finished = 0;
  if (CHECK && !(mode & PROX_FINAL)) {
    double nx = 0, nz = 0, nrp = 0, nrd = 0, nPx = 0, ny = 0, nq = 0;
    for (int j = 0; j < nslot; ++j) {
      const int t = j * RES_NT + tid;
      if (t >= n_slice) break;
      const int64_t gi = i_beg + t;
      const double T = Ts[t], w0 = ws[t];
      const double tr = trade(t, gi, T, w0, p.invd[gi]);
      const double z = w0 + tr;
      const double y = T + lam_b - tr * (cg * p.d[gi]);
      const double x = p.xs[rowp + gi], pq = p.pxq[rowp + gi];
      const double qi = p.q ? p.q[rowp + gi] : -p.mu[row + gi];
      nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
      nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq - qi)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qi));
      if (!(z == z) || !(x == x) || !(T == T) || !(pq == pq)) nrp = INFINITY;     // fmax drops NaN: poison explicitly
    }
    double val[7] = {nx, nz, nrp, nrd, nPx, ny, nq};
    src.template reduce<7, 1>(val, nullptr);
    const double rp = val[2] / fmax(fmax(val[0], val[1]), 1e-300);
    const double rd = val[3] / fmax(fmax(val[4], fmax(val[5], val[6])), 1e-300);
    const bool bad = !(rp < INFINITY) || !(rd < INFINITY) || !(alpha == alpha) || !(beta == beta);
    const bool conv = !bad && rp <= p.eps && rd <= p.eps && !rs.capped;            // never certify on an unfinished root find
    if (tid == 0 && rank == 0) {
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_PRIMAL] = rp;
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_DUAL] = rd;
    }
    if (conv || bad) {
      finished = 1;
      if (tid == 0 && rank == 0) p.ap.conv[a] = bad ? -1 : 1;
    } else if (p.adapt && p.iter >= PRISM_ADAPT_START && p.iter - nadapt_prev >= PRISM_ADAPT_EVERY) {
      const double ratio = sqrt(rp / fmax(rd, 1e-300));
      if (ratio > 3.0 || ratio < 1.0 / 3.0) {
        c_new = c * fmin(fmax(ratio, 0.2), 5.0);
        if (tid == 0 && rank == 0) { p.ap.c[a] = c_new; p.ap.refactor[a] = 1; }
      }
      if (tid == 0 && rank == 0) p.ap.nadapt[a] = p.iter;
    }
  }
  if (mode & PROX_FINAL) finished = 1;

  // ---- C. outputs of the slice
  {
    const double cgn = c_new * gam, igc = 1.0 / (gam * (1.0 + c_new)), icgn = 1.0 / cgn;
    const bool rescale = c_new != c;
    for (int j = 0; j < nslot; ++j) {
      const int t = j * RES_NT + tid;
      if (t >= n_slice) break;
      const int64_t gi = i_beg + t;
      const double T = Ts[t], w0 = ws[t], iv = p.invd[gi];
      const double tr = trade(t, gi, T, w0, iv);
      const double z = w0 + tr;
      if (CHECK) p.w_out[row + gi] = z;                    // kept if the account finishes here
      if (finished) continue;
      const double di = p.d[gi];
      const double y = T + lam_b - tr * (cg * di);         // rho_old (v - z): unchanged by a rho change
      if (rescale) p.v[rowp + gi] = z + y * iv * icgn;     // v' = z + y / rho_new
      const double qi = p.q ? p.q[rowp + gi] : -p.mu[row + gi];
      const double r = cgn * di * z - y - qi;
      const double rt = r * iv * igc;                      // M_i = gamma d_i (1 + c)
      p.rt[rowp + gi] = rt;
      p.cc[rowp + gi] = rt - z;
    }
  }
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
