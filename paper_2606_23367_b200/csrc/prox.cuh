// prox.cuh - H4 fused proximal / projection kernel, one CTA per account.
//
// z-update of the splitting, in trade space t = z - w0, u = v - w0, rho_i = c gamma d_i:
//
//   minimise  sum_i [ rho_i/2 (t_i - u_i)^2 + (kappa + c_buy) (t_i)_+ + kappa (-t_i)_+ + psi_i((-t_i)_+) ]
//   s.t.      sum_i t_i = 1 - sum_i w0_i          (budget hyperplane, Eq. (1) row 1)
//             lo_i <= w0_i + t_i <= hi_i          (box, exclusions as lo = hi = 0)
//             sum_i |t_i| <= tau                  (turnover budget, D_a = I)
//
// With multipliers nu (budget) and theta >= 0 (turnover), alpha = nu + theta and beta = nu - theta, buys depend on
// alpha only and sells on beta only ("L1 turnover split", BASELINE.json:north_star):
//   buy_i(alpha)  = clip((rho_i u_i - kappa - c_buy - alpha) / rho_i, bl_i, bh_i)
//   sell_i(beta)  = clip(sum_l clip((beta - rho_i u_i - kappa - s_il)/rho_i - Q_{i,l-1}, 0, q_il), sl_i, sh_i)
// so the two coupled constraints become:  theta = 0: one monotone scalar equation  P(nu) - R(nu) = b;
// cap active: two independent monotone equations  P(alpha) = (tau + b)/2,  R(beta) = (tau - b)/2.
// Each is continuous piecewise linear; solved by safeguarded Newton (bracketed, exact on the final linear piece),
// warm-started from the previous iteration.  All trial evaluations are block-wide reductions in this CTA.
//
// Group bands (Eq. (1) row 3 with A_a = group indicators) are handled in the same projection: with
// multipliers lambda_g (> 0: upper band active, < 0: lower band active) the thresholds of an asset of group g
// become alpha + lambda_g and beta + lambda_g.  For fixed lambda the (alpha, beta) equations keep their form; the
// group sums S_g(lambda_g) (with alpha, beta re-solved) are monotone, so violated / active groups are fixed one
// at a time by a bracketed scalar Newton iteration on lambda_g (Gauss-Seidel over groups, usually 0 or 1 group).
// Putting ALL polyhedral constraints into this projection (instead of a consensus block in the x-update) is what
// makes the splitting converge in a few hundred iterations: a consensus row's dual moves at rate
// (#moving assets)/(#assets in the row) per iteration ("why the bands live in the prox").
//
// The same kernel then emits what the x-update needs (r~ = M^-1 r, c = r~ - z, per-group sums of r~), and on check
// iterations the scaled residuals, the convergence mask and the per-account rho adaptation.
#pragma once
#include "common.cuh"

struct ProxArgs {
  int64_t N, ldw;           // ldw: leading dimension of the owned A x N arrays (v, rt, cc, xs, pxq, q)
  int32_t A, G, kp, max_lots;
  int64_t ldv;
  // borrowed data
  const double *mu, *q, *w0, *gamma, *lo, *hi, *hi_full, *tau, *kappa, *c_buy, *lot_slope, *lot_width;
  const uint8_t *excl, *lot_count, *group_id;
  const double* invd;
  const double* d;
  // iterate
  double *v, *rt, *cc;
  const double *xs, *pxq;
  const double *band_lo, *band_hi;
  double *lamG;             // A x G band multipliers (warm start, persists across iterations)
  const double *gw0;        // A x G group sums of w0
  AccountParams ap;
  double* w_out;
  double* duals;
  double* resid;
  int32_t* counters;
  // settings
  double eps, eps_abs;      // converged when r <= eps_abs + eps * scale for both residuals
  int32_t adapt, iter;
  int32_t sample_until;    // streaming form: plain launches of iterations < sample_until (bands still out) use the sampled root find
  int32_t adapt_start, adapt_every;   // first iteration at which an account's rho may be adapted; minimum iterations between two
  double win_mult;         // next window = win_mult x (movement of the thresholds in this launch)
  double win_ratio;        // streaming pass: its (wide) window = win_ratio x the solve's (tight) window
  int32_t band_start;      // streaming form: group bands join the projection after this iteration (their multipliers are 0 before)
  int32_t band_wide;       // 1: the launch in which the bands join runs with an infinite window
  int32_t band_ramp;       // ... with limits widened by slack_a (1 - (iter - band_start) / band_ramp) for band_ramp iterations
  // streaming form (prox_fast.cuh): per-warp live lists, their compacted copy, fixed-point bins of the dead assets
  struct LiveEnt* lraw;    // [A][S * 8][capw]
  struct LiveEnt* lcomp;   // [A][ldc]
  int32_t* lcnt;           // [A][S * 8]
  unsigned long long* cbin;// [A][2 max(G, 1)]  buys, sells per group in units of 2^-60 (zero between launches)
  double* chkp;            // [A][S][8] residual terms of the dead assets per slice (check iterations)
  int32_t* lflag;          // [A] 1: the account takes the generic path in k_prox_root
  int32_t S, capw;         // slices per account; capacity of one warp's list
  int64_t slice_len, ldc;  // assets per slice (multiple of 512); entries per account in lcomp
  // cluster-resident form (prox_res.cuh): CTAs per account (cluster size) and assets per CTA (multiple of 256)
  int32_t res_C, res_SL;
};

enum { PROX_CHECK = 1, PROX_FINAL = 2 };

// Per-element constants of one launch, in "threshold space":  T = rho u - (kappa + c_buy),  Delta = 2 kappa + c_buy:
//   buy_i(a)  = bl + clamp((T - a) / rho - bl, 0, wB)            a  = alpha + lambda_g
//   sell_i(b) = sl + clamp((b - Delta - T) / rho - sl, 0, wS)    b  = beta + lambda_g
// (with lots: sum over lots of clamp((b - Delta - s_l - T)/rho - Q_{l-1}, 0, q_l), clipped to [sl, min(sl + wS, Q_L)]).
struct ElemConst {
  double T, ir, bl, wB, sl, wS, w0;      // ir = 1 / rho_i; buy range [bl, bl + wB]; sell range [sl, sl + wS]
  double d, qv;                          // d_i and q_ai: filled by for_each_all only (check / output passes)
};

__device__ __forceinline__ void elem_ranges(ElemConst& e, double lo, double hi) {
  const double bh = fmax(hi - e.w0, 0.0), sh = fmax(e.w0 - lo, 0.0);
  e.bl = fmax(lo - e.w0, 0.0);
  e.sl = fmax(e.w0 - hi, 0.0);
  e.wB = bh - e.bl;
  e.wS = sh - e.sl;
}

// buy amount at threshold a; mv = 1/rho_i if strictly inside its range (|slope| of the piece), else 0
__device__ __forceinline__ double buy_amt(const ElemConst& e, double a, double& mv) {
  const double tb = (e.T - a) * e.ir - e.bl;
  mv = 0.0;
  if (tb <= 0.0) return e.bl;
  if (tb >= e.wB) return e.bl + e.wB;
  mv = e.ir;
  return e.bl + tb;
}

template <bool LOTS>
__device__ __forceinline__ double sell_amt(const ElemConst& e, double bd, const double* slope, const double* width,
                                           int nl, double& mv) {   // bd = beta + lambda_g - Delta
  mv = 0.0;
  if (LOTS && nl > 0) {
    // the asset's whole lot row (4 slopes, 4 widths: two 32-byte rows, 16-byte aligned by the ABI) in ONE round of loads -
    // a loop that fetches lot l only after lot l - 1 has been accounted for is a chain of up to eight global-load latencies
    // per live asset per pass (14% of the lots kernel's stall samples, profiles/r2_kernels_ncu_full.md)
    const double2 s01 = *(const double2*)slope, s23 = *(const double2*)(slope + 2);
    const double2 w01 = *(const double2*)width, w23 = *(const double2*)(width + 2);
    const double sl4[PRISM_MAX_LOTS] = {s01.x, s01.y, s23.x, s23.y}, wd4[PRISM_MAX_LOTS] = {w01.x, w01.y, w23.x, w23.y};
    double raw = 0.0, Q = 0.0, inside = 0.0;
#pragma unroll
    for (int l = 0; l < PRISM_MAX_LOTS; ++l) {
      if (l < nl) {
        const double r = (bd - sl4[l] - e.T) * e.ir - Q;
        const double ql = wd4[l];
        if (r > 0.0 && r < ql) inside = 1.0;
        raw += fmin(fmax(r, 0.0), ql);
        Q += ql;
      }
    }
    const double sh = fmin(e.sl + e.wS, Q);
    if (inside > 0.0 && raw > e.sl && raw < sh) mv = e.ir;
    return fmin(fmax(raw, e.sl), sh);
  }
  const double ts = (bd - e.T) * e.ir - e.sl;
  if (ts <= 0.0) return e.sl;
  if (ts >= e.wS) return e.sl + e.wS;
  mv = e.ir;
  return e.sl + ts;
}

// One bracketed Newton step on a continuous piecewise-linear monotone function.
// dir = +1: g increasing in x, -1: decreasing.  slope = |g'| at x (0 on a flat piece).  Brackets may be infinite
// (lazy): then a step that cannot use Newton reports need_bracket instead.  With finite brackets such a step asks
// for a SECTION pass (sect = 1): the caller evaluates the function at PROX_KSEC points of the bracket in one pass
// over the assets (prox_eval_multi) and root_place() shrinks the bracket to the sub-interval that holds the root.
#define PROX_KSEC 8
struct Root1D {
  double x, lo, hi;
  int done, sect;
};
__device__ __forceinline__ bool root_step(Root1D& r, double g, double slope, double target, int dir, double tol) {
  if (r.done) return false;
  const double diff = g - target;
  if (fabs(diff) <= tol) { r.done = 1; return false; }
  const bool too_big = (dir > 0) ? (diff > 0.0) : (diff < 0.0);   // x lies right of the root
  if (too_big) r.hi = r.x; else r.lo = r.x;
  const double xn = (slope > 0.0) ? r.x - (double)dir * diff / slope : NAN;
  if (!(xn > r.lo && xn < r.hi)) {
    if (!(r.lo > -INFINITY) || !(r.hi < INFINITY)) return true;   // needs finite brackets
    const double mid = 0.5 * (r.lo + r.hi);
    if (!(mid > r.lo && mid < r.hi)) { r.done = 1; return false; } // bracket exhausted (adjacent doubles)
    r.sect = 1;
    return false;
  }
  if (xn == r.x) { r.done = 1; return false; }
  r.x = xn;
  return false;
}
// f[k] = function at x0 + k dx, k = 0 .. PROX_KSEC-1 (points strictly inside the bracket, ascending): new bracket =
// the sub-interval that holds the root, new x = secant point of its ends (midpoint where an end value is unknown).
__device__ __forceinline__ void root_place(Root1D& r, const double* f, double x0, double dx, double target, int dir) {
  int kr = PROX_KSEC;
  for (int k = PROX_KSEC - 1; k >= 0; --k) {
    const double diff = f[k] - target;
    if ((dir > 0) ? (diff > 0.0) : (diff < 0.0)) kr = k;          // x_k lies right of the root (monotone => a suffix)
  }
  const double lo = kr == 0 ? r.lo : x0 + (kr - 1) * dx, hi = kr == PROX_KSEC ? r.hi : x0 + kr * dx;
  double x = 0.5 * (lo + hi);
  if (kr > 0 && kr < PROX_KSEC) {
    const double flo = f[kr - 1], fhi = f[kr];
    if (fhi != flo) { const double xs = lo + (target - flo) / (fhi - flo) * (hi - lo); if (xs > lo && xs < hi) x = xs; }
  }
  r.lo = lo; r.hi = hi; r.sect = 0;
  if (!(x > lo && x < hi)) { r.done = 1; x = lo; }
  r.x = x;
}

// ---------------------------------------------------------------------------------------------- element sources
// A source enumerates the assets the root find has to look at (for_each / for_each_uniform) and supplies the
// constant parts of the sums that it does not enumerate: cP(), cR() (total buys / sells of the assets whose trade
// cannot change inside the current window) and the same per group, cPg(g), cRg(g).

// Generic source: every pass re-reads the account from global memory (any N, lots, per-asset caps).
template <bool LOTS>
struct SrcGlobal {
  const ProxArgs& p;
  int64_t row, rowp;
  double cg, icg, lo_a, hi_a, lam_b;
  __device__ SrcGlobal(const ProxArgs& p_, int a, double cg_, double lo, double hi, double lam_b_)
      : p(p_), row((int64_t)a * p_.N), rowp((int64_t)a * p_.ldw), cg(cg_), icg(1.0 / cg_), lo_a(lo), hi_a(hi), lam_b(lam_b_) {}
  __device__ __forceinline__ void load(int64_t i, ElemConst& e, int& g, int& nl, const double*& sl, const double*& wd) const {
    const int64_t idx = row + i;
    e.w0 = p.w0[idx];
    e.T = (p.v[rowp + i] - e.w0) * (cg * p.d[i]) - lam_b;
    e.ir = p.invd[i] * icg;
    double lo = lo_a, hi = p.hi_full ? p.hi_full[idx] : hi_a;
    if (p.excl && p.excl[idx]) { lo = 0.0; hi = 0.0; }
    elem_ranges(e, lo, hi);
    g = p.G ? p.group_id[i] : 0;
    nl = 0; sl = nullptr; wd = nullptr;
    if (LOTS) { nl = p.lot_count[idx]; sl = p.lot_slope + idx * PRISM_MAX_LOTS; wd = p.lot_width + idx * PRISM_MAX_LOTS; }
  }
  template <class F>
  __device__ __forceinline__ void for_each(F f) const {          // f(i, e, g, nl, sl, wd)
    for (int64_t i = threadIdx.x; i < p.N; i += blockDim.x) {
      ElemConst e; int g, nl; const double *sl, *wd;
      load(i, e, g, nl, sl, wd);
      f(i, e, g, nl, sl, wd);
    }
  }
  template <class F>
  __device__ __forceinline__ void for_each_uniform(F f) const {  // f(valid, i, e, g, nl, sl, wd), warp-uniform trip count
    for (int64_t i0 = 0; i0 < p.N; i0 += blockDim.x) {
      const int64_t i = i0 + threadIdx.x;
      const bool valid = i < p.N;
      ElemConst e; int g = 0, nl = 0; const double *sl = nullptr, *wd = nullptr;
      if (valid) load(i, e, g, nl, sl, wd);
      f(valid, i, e, g, nl, sl, wd);
    }
  }
  template <class F>
  __device__ __forceinline__ void for_each_all(F f) const {
    for (int64_t i = threadIdx.x; i < p.N; i += blockDim.x) {
      ElemConst e; int g, nl; const double *sl, *wd;
      load(i, e, g, nl, sl, wd);
      e.d = p.d[i];
      e.qv = p.q ? p.q[rowp + i] : -p.mu[row + i];
      f(i, e, g, nl, sl, wd);
    }
  }
  // block-wide reduction used by the generic evaluation routines (a cluster-resident source reduces over its cluster)
  template <int NV, int OP>
  __device__ __forceinline__ void reduce(double (&val)[NV], double* scratch) const { block_reduce<NV, OP>(val, scratch); }
  __device__ __forceinline__ void classify(double, double, const double*, double, int*) {}
  __device__ __forceinline__ bool window_ok(double, double, const double*) const { return true; }
  __device__ __forceinline__ double cP() const { return 0.0; }
  __device__ __forceinline__ double cR() const { return 0.0; }
  __device__ __forceinline__ double cPg(int) const { return 0.0; }
  __device__ __forceinline__ double cRg(int) const { return 0.0; }
};

// Shared-memory source: T and w0 of the whole account (2 x 8 B x N) plus a class byte and the group id per asset
// stay in shared memory for the kernel, so a trial evaluation touches no HBM: only 1/d_i (shared by all accounts,
// L2 resident).  No lots, no per-asset caps.  Used when the streaming form (prox_fast.cuh) does not apply (N not a multiple of 16) and N is small enough.
//
// Live list.  Most assets sit on the kink (no trade) and stay there while the thresholds move a little, so the
// root-finding passes only visit the assets that can trade for thresholds inside a WINDOW around the warm start:
// a regular asset is dead if  T <= (alpha_w + lambda_w,g) - W  and  T + Delta >= (beta_w + lambda_w,g) + W;  then its
// buy and sell amounts are exactly 0 whenever |alpha - alpha_w|, |beta - beta_w|, |lambda_g - lambda_w,g| <= W / 2.
// The solve runs on the live list; if its result leaves the window it is repeated with W = inf (all assets).
// The list is compacted in (thread, slot) order by a block scan, so every sum keeps a fixed order (deterministic).
struct SrcSmem {
  const ProxArgs& p;
  int64_t row, rowp;
  double icg, lo_a, hi_a, Delta;
  double *Ts, *ws;
  uint8_t *cls, *gid;      // cls: 0 regular (lo <= w0 <= hi, not excluded), 1 excluded, 2 outside the box
  uint16_t* live;
  int n_live;
  double aw, bw, W;        // warm-start thresholds and window
  const double* lam_w;     // warm-start band multipliers (global, G entries)
  __device__ SrcSmem(const ProxArgs& p_, int a, double cg, double lo, double hi, double lam_b, double Delta_, double* smem)
      : p(p_), row((int64_t)a * p_.N), rowp((int64_t)a * p_.ldw), icg(1.0 / cg), lo_a(lo), hi_a(hi), Delta(Delta_), Ts(smem),
        ws(smem + p_.N), cls((uint8_t*)(smem + 2 * p_.N)), gid((uint8_t*)(smem + 2 * p_.N) + p_.N),
        live((uint16_t*)((uint8_t*)(smem + 2 * p_.N) + 2 * p_.N)), n_live(0), aw(0), bw(0), W(INFINITY), lam_w(nullptr) {
    constexpr int CB = 8;                              // loads of CB slots are issued together (memory-level parallelism)
    const int64_t nt = blockDim.x;
    for (int64_t i0 = threadIdx.x; i0 < p.N; i0 += CB * nt) {
      double v8[CB], w8[CB], d8[CB]; uint8_t e8[CB], g8[CB];
#pragma unroll
      for (int u = 0; u < CB; ++u) {
        const int64_t i = i0 + u * nt;
        if (i < p.N) {
          w8[u] = p.w0[row + i]; v8[u] = p.v[rowp + i]; d8[u] = p.d[i];
          e8[u] = p.excl ? p.excl[row + i] : 0; g8[u] = p.G ? p.group_id[i] : 0;
        }
      }
#pragma unroll
      for (int u = 0; u < CB; ++u) {
        const int64_t i = i0 + u * nt;
        if (i < p.N) {
          ws[i] = w8[u];
          Ts[i] = (v8[u] - w8[u]) * (cg * d8[u]) - lam_b;
          cls[i] = e8[u] ? 1 : ((w8[u] >= lo && w8[u] <= hi) ? 0 : 2);
          gid[i] = g8[u];
        }
      }
    }
  }
  // (Re)build the live list for the window W around (aw_, bw_, lam_w_).  scratch: >= 64 ints of shared memory.
  __device__ void classify(double aw_, double bw_, const double* lam_w_, double W_, int* scratch) {
    aw = aw_; bw = bw_; lam_w = lam_w_; W = W_;
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, wid = tid >> 5, nw = (nt + 31) >> 5;
    const bool all = !(W < INFINITY);
    auto is_live = [&](int64_t i) -> bool {
      if (all || cls[i] != 0) return true;
      const double lg = p.G ? lam_w[gid[i]] : 0.0;
      const double T = Ts[i];
      return !(T <= aw + lg - W && T + Delta >= bw + lg + W);
    };
    // index-ordered compaction (keeps shared-memory and global accesses of the live passes coalesced):
    // per (slot, warp) counts by ballot -> serial exclusive scan of the small table -> ballot again and write
    const int nslot = (int)((p.N + nt - 1) / nt);
    __syncthreads();                                   // scratch may still be in use by an earlier reduction
    for (int sl = 0; sl < nslot; ++sl) {
      const int64_t i = (int64_t)sl * nt + tid;
      const unsigned m = __ballot_sync(0xffffffffu, i < p.N && is_live(i));
      if (lane == 0) scratch[sl * nw + wid] = __popc(m);
    }
    __syncthreads();
    if (tid == 0) {
      int run = 0;
      for (int q = 0; q < nslot * nw; ++q) { const int t = scratch[q]; scratch[q] = run; run += t; }
      scratch[nslot * nw] = run;
    }
    __syncthreads();
    for (int sl = 0; sl < nslot; ++sl) {
      const int64_t i = (int64_t)sl * nt + tid;
      const bool lv = i < p.N && is_live(i);
      const unsigned m = __ballot_sync(0xffffffffu, lv);
      if (lv) live[scratch[sl * nw + wid] + __popc(m & ((1u << lane) - 1u))] = (uint16_t)i;
    }
    n_live = scratch[nslot * nw];
    __syncthreads();
  }
  // block-wide reduction used by the generic evaluation routines (a cluster-resident source reduces over its cluster)
  template <int NV, int OP>
  __device__ __forceinline__ void reduce(double (&val)[NV], double* scratch) const { block_reduce<NV, OP>(val, scratch); }
  __device__ __forceinline__ bool window_ok(double al, double be, const double* lamS) const {
    if (!(W < INFINITY)) return true;
    bool ok = fabs(al - aw) <= 0.5 * W && fabs(be - bw) <= 0.5 * W;
    for (int g = 0; g < p.G; ++g) ok = ok && fabs(lamS[g] - lam_w[g]) <= 0.5 * W;
    return ok;
  }
  __device__ __forceinline__ void load(int64_t i, ElemConst& e, int& g) const {
    e.w0 = ws[i]; e.T = Ts[i];
    e.ir = p.invd[i] * icg;
    const int c = cls[i];
    g = gid[i];
    if (c == 0) { e.bl = 0.0; e.sl = 0.0; e.wB = hi_a - e.w0; e.wS = e.w0 - lo_a; }
    else elem_ranges(e, c == 1 ? 0.0 : lo_a, c == 1 ? 0.0 : hi_a);
  }
  // live assets only (root-finding passes)
  template <class F>
  __device__ __forceinline__ void for_each(F f) const {
#pragma unroll 2
    for (int j = threadIdx.x; j < n_live; j += blockDim.x) {
      const int64_t i = live[j];
      ElemConst e; int g;
      load(i, e, g);
      f(i, e, g, 0, (const double*)nullptr, (const double*)nullptr);
    }
  }
  template <class F>
  __device__ __forceinline__ void for_each_uniform(F f) const {
    for (int j0 = 0; j0 < n_live; j0 += blockDim.x) {
      const int j = j0 + threadIdx.x;
      const bool valid = j < n_live;
      const int64_t i = valid ? live[j] : 0;
      ElemConst e; int g = 0;
      if (valid) load(i, e, g);
      f(valid, i, e, g, 0, (const double*)nullptr, (const double*)nullptr);
    }
  }
  // every asset (check and output passes), loads batched (shared memory, 1/d, d and q of PB slots together)
  template <class F>
  __device__ __forceinline__ void for_each_all(F f) const {
    constexpr int PB = 6;
    const int64_t nt = blockDim.x;
    for (int64_t i0 = threadIdx.x; i0 < p.N; i0 += PB * nt) {
      double T4[PB], w4[PB], iv4[PB], d4[PB], q4[PB]; int c4[PB], g4[PB];
#pragma unroll
      for (int u = 0; u < PB; ++u) {
        const int64_t i = i0 + u * nt;
        if (i < p.N) {
          T4[u] = Ts[i]; w4[u] = ws[i]; iv4[u] = p.invd[i]; d4[u] = p.d[i]; c4[u] = cls[i]; g4[u] = gid[i];
          q4[u] = p.q ? p.q[rowp + i] : -p.mu[row + i];
        }
      }
#pragma unroll
      for (int u = 0; u < PB; ++u) {
        const int64_t i = i0 + u * nt;
        if (i < p.N) {
          ElemConst e;
          e.w0 = w4[u]; e.T = T4[u]; e.ir = iv4[u] * icg; e.d = d4[u]; e.qv = q4[u];
          if (c4[u] == 0) { e.bl = 0.0; e.sl = 0.0; e.wB = hi_a - e.w0; e.wS = e.w0 - lo_a; }
          else elem_ranges(e, c4[u] == 1 ? 0.0 : lo_a, c4[u] == 1 ? 0.0 : hi_a);
          f(i, e, g4[u], 0, (const double*)nullptr, (const double*)nullptr);
        }
      }
    }
  }
  __device__ __forceinline__ double cP() const { return 0.0; }
  __device__ __forceinline__ double cR() const { return 0.0; }
  __device__ __forceinline__ double cPg(int) const { return 0.0; }
  __device__ __forceinline__ double cRg(int) const { return 0.0; }
};

// Shared-memory work areas of the root find (static in the slow kernels, carved from dynamic memory in the fast one).
struct ProxShared {
  double* scratch;   // 12 * 32
  double* gbin;      // nwarps * G   per-warp group bins (deterministic accumulation)
  double* lamS;      // G            band multipliers being solved for
  double* gsum;      // G
  int* selS;         // 2
  const double *band_lo, *band_hi, *gw0;   // G each, this account's rows (global, or shared-memory copies)
};

// One pass over the account: totals P, R and their slopes at thresholds (al, bd + Delta) shifted by the group
// multipliers, plus the same four sums restricted to up to two selected groups s1, s2 (-1 = none).
// out[0..3] = P, R, sP, sR;  out[4..7] = group s1;  out[8..11] = group s2.   Not inlined: it is called from many places.
template <bool LOTS, class Src>
__device__ __noinline__ void prox_eval(const Src& src, const double* lamS, int G, double al, double bd, int s1, int s2,
                                       double* scratch, double* out) {
  double lP = 0, lR = 0, lsP = 0, lsR = 0, x[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  src.for_each([&](int64_t, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
    double mvb, mvs;
    const double lg = G ? lamS[g] : 0.0;
    const double pb = buy_amt(e, al + lg, mvb);
    const double ps = sell_amt<LOTS>(e, bd + lg, sl, wd, nl, mvs);
    lP += pb; lR += ps; lsP += mvb; lsR += mvs;
    if (g == s1) { x[0] += pb; x[1] += ps; x[2] += mvb; x[3] += mvs; }
    if (g == s2) { x[4] += pb; x[5] += ps; x[6] += mvb; x[7] += mvs; }
  });
  if (s1 >= 0 || s2 >= 0) {
    double val[12] = {lP, lR, lsP, lsR, x[0], x[1], x[2], x[3], x[4], x[5], x[6], x[7]};
    src.template reduce<12, 0>(val, scratch);
#pragma unroll
    for (int q = 0; q < 12; ++q) out[q] = val[q];
    if (s1 >= 0) { out[4] += src.cPg(s1); out[5] += src.cRg(s1); }
    if (s2 >= 0) { out[8] += src.cPg(s2); out[9] += src.cRg(s2); }
  } else {
    double val[4] = {lP, lR, lsP, lsR};
    src.template reduce<4, 0>(val, scratch);
#pragma unroll
    for (int q = 0; q < 4; ++q) out[q] = val[q];
  }
  out[0] += src.cP(); out[1] += src.cR();
}

// Section pass: buys at the PROX_KSEC thresholds a0 + k da and sells at b0 + k db (b = beta - Delta), one pass.
template <bool LOTS, class Src>
__device__ __noinline__ void prox_eval_multi(const Src& src, const double* lamS, int G, double a0, double da, double b0,
                                             double db, double* scratch, double* outP, double* outR) {
  double sp[PROX_KSEC], sr[PROX_KSEC];
#pragma unroll
  for (int k = 0; k < PROX_KSEC; ++k) { sp[k] = 0.0; sr[k] = 0.0; }
  src.for_each([&](int64_t, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
    const double lg = G ? lamS[g] : 0.0;
#pragma unroll
    for (int k = 0; k < PROX_KSEC; ++k) {
      double mvb, mvs;
      sp[k] += buy_amt(e, a0 + k * da + lg, mvb);
      sr[k] += sell_amt<LOTS>(e, b0 + k * db + lg, sl, wd, nl, mvs);
    }
  });
  const double cP = src.cP(), cR = src.cR();
#pragma unroll
  for (int q0 = 0; q0 < PROX_KSEC; q0 += 8) {
    double val[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) val[q] = sp[q0 + q];
    src.template reduce<8, 0>(val, scratch);
#pragma unroll
    for (int q = 0; q < 8; ++q) outP[q0 + q] = val[q] + cP;
#pragma unroll
    for (int q = 0; q < 8; ++q) val[q] = sr[q0 + q];
    src.template reduce<8, 0>(val, scratch);
#pragma unroll
    for (int q = 0; q < 8; ++q) outR[q0 + q] = val[q] + cR;
  }
}

// Range of the breakpoints in threshold space: out = {a_min, a_max, b_min, b_max} (only when bisection is needed).
template <bool LOTS, class Src>
__device__ __noinline__ void prox_brackets(const Src& src, double Delta, double* scratch, double* out) {
  double x4 = INFINITY, x5 = -INFINITY, x6 = INFINITY, x7 = -INFINITY;
  src.for_each([&](int64_t, const ElemConst& e, int, int nl, const double* sl, const double* wd) {
    const double rho = 1.0 / e.ir;
    if (e.wB > 0.0) { x4 = fmin(x4, e.T - rho * (e.bl + e.wB)); x5 = fmax(x5, e.T - rho * e.bl); }
    double sh = e.sl + e.wS, s_first = 0.0, s_last = 0.0;
    if (LOTS && nl > 0) { double Q = 0; for (int l = 0; l < nl; ++l) Q += wd[l]; sh = fmin(sh, Q); s_first = sl[0]; s_last = sl[nl - 1]; }
    if (sh > e.sl) { x6 = fmin(x6, e.T + Delta + s_first + rho * e.sl); x7 = fmax(x7, e.T + Delta + s_last + rho * sh); }
  });
  double val[4] = {-x4, x5, -x6, x7};          // min via max of the negation: one uniform reduction
  src.template reduce<4, 1>(val, scratch);
  out[0] = -val[0]; out[1] = val[1]; out[2] = -val[2]; out[3] = val[3];
}

// Sums of the trades per group at the final thresholds -> gsum[g] = gw0[g] + sum (deterministic binned pass).
template <bool LOTS, class Src>
__device__ __noinline__ void prox_group_sums(const Src& src, const double* lamS, int G, double al, double bd,
                                             const double* gw0, double* gbin, double* gsum) {
  const int tid = threadIdx.x, nt = blockDim.x, nw = (nt + 31) >> 5;
  for (int g = tid; g < nw * G; g += nt) gbin[g] = 0.0;
  __syncthreads();
  src.for_each_uniform([&](bool valid, int64_t, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
    double t = 0.0;
    if (valid) {
      double mvb, mvs;
      t = buy_amt(e, al + lamS[g], mvb) - sell_amt<LOTS>(e, bd + lamS[g], sl, wd, nl, mvs);
    }
    warp_group_add(gbin, G, valid ? g : 0, t, valid);
  });
  __syncthreads();
  for (int g = tid; g < G; g += nt) gsum[g] = gw0[g] + group_total(gbin, G, g) + (src.cPg(g) - src.cRg(g));
  __syncthreads();
}

// Scaled residuals of the splitting (reading R13) from the stored x and P x + q: out = {r_p, r_d, tolerance met}.
template <bool LOTS, class Src>
__device__ __noinline__ void prox_check(const ProxArgs& p, const Src& src, const double* lamS, int a, double al, double bd,
                                        double lam_b, double cg, double* scratch, double* out) {
  const int G = p.G;
  const int64_t rowp = (int64_t)a * p.ldw;
  double nx = 0, nz = 0, nrp = 0, nrd = 0, nPx = 0, ny = 0, nq = 0;
  src.for_each_all([&](int64_t i, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
    double mvb, mvs;
    const double lg = G ? lamS[g] : 0.0;
    const double tr = buy_amt(e, al + lg, mvb) - sell_amt<LOTS>(e, bd + lg, sl, wd, nl, mvs);
    const double z = e.w0 + tr;
    const double y = e.T + lam_b - tr * (cg * e.d);     // rho (v - z) = rho u - rho t
    const double x = p.xs[rowp + i], pq = p.pxq[rowp + i];
    const double qi = e.qv;
    nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
    nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq - qi)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qi));
    if (!(z == z) || !(x == x) || !(e.T == e.T)) nrp = INFINITY;     // fmax drops NaN: poison explicitly
  });
  double val[7] = {nx, nz, nrp, nrd, nPx, ny, nq};
  block_reduce<7, 1>(val, scratch);
  out[0] = val[2] / fmax(fmax(val[0], val[1]), 1e-300);
  out[1] = val[3] / fmax(fmax(val[4], fmax(val[5], val[6])), 1e-300);
  out[2] = (val[2] <= p.eps_abs + p.eps * fmax(val[0], val[1]) && val[3] <= p.eps_abs + p.eps * fmax(val[4], fmax(val[5], val[6]))) ? 1.0 : 0.0;
}

// Output pass: either the returned weights (finished) or what the x-update needs: r~ = M^-1 r, c = r~ - z,
// and v re-expressed in the new rho when it changed.  (e.T, e.ir refer to the old rho.)
template <bool LOTS, class Src>
__device__ __noinline__ void prox_output(const ProxArgs& p, const Src& src, const double* lamS, int a, double al, double bd,
                                         double lam_b, double gam, double c_old, double c_new, int finished) {
  const int G = p.G;
  const int64_t row = (int64_t)a * p.N, rowp = (int64_t)a * p.ldw;
  const double cg = c_old * gam, cgn = c_new * gam, igc = 1.0 / (gam * (1.0 + c_new)), icgn = 1.0 / cgn;
  const bool rescale = c_new != c_old;
  src.for_each_all([&](int64_t i, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
    double mvb, mvs;
    const double lg = G ? lamS[g] : 0.0;
    const double tr = buy_amt(e, al + lg, mvb) - sell_amt<LOTS>(e, bd + lg, sl, wd, nl, mvs);
    const double z = e.w0 + tr;
    if (finished) { p.w_out[row + i] = z; return; }
    const double di = e.d, dinv = e.ir * cg;               // e.ir = 1 / (c_old gamma d_i)
    const double y = e.T + lam_b - tr * (cg * di);         // rho_old (v - z): unchanged by a rho change
    if (rescale) p.v[rowp + i] = z + y * dinv * icgn;      // v' = z + y / rho_new
    const double qi = e.qv;
    const double r = cgn * di * z - y - qi;
    const double rt = r * dinv * igc;                      // M_i = gamma d_i (1 + c)
    p.rt[rowp + i] = rt;
    p.cc[rowp + i] = rt - z;
  });
}

// ------------------------------------------------------------------------------------------------ the root find
struct RootState {
  double alpha, beta;    // in: warm start; out: thresholds  nu + theta,  nu - theta
  int amode;             // 0: turnover cap inactive (alpha == beta), 1: active
  int n_eval;            // trial evaluations (passes over the source) spent
  int nobands;           // in: 1 = solve with every band multiplier fixed at 0 (band ramp of the first iterations)
  int max_rounds;        // in: Gauss-Seidel rounds over the bands the nested solve may take before it reports capped = 2
  int capped;            // out: 2 = the Gauss-Seidel rounds ran out before every band held (the caller polishes with the joint
                         // Newton iteration and calls again); 1 = the evaluation budget ran out (PROX_EVAL_CAP): the thresholds are the last iterate, NOT a
                         // solution.  The caller may use them for a plain iteration (an inexact prox) but must not
                         // certify convergence with them.
};
// Budget of trial evaluations of one nested robust solve: its worst case (Gauss-Seidel rounds x bracketed steps x inner
// root finds) is ~1e5 passes, and one account that wanders there holds its whole launch.  Regular solves need <= ~300;
// the budget only bounds the damage of a pathological one (readings: robust root find).
#ifndef PROX_EVAL_CAP
#define PROX_EVAL_CAP 2000
#endif

// Solves for (alpha, beta, lambda_g) of account a over the assets of `src` (see the header of this file).
// b: budget in trade space, tau: turnover cap (inf = none), Delta = 2 kappa + c_buy.  sh.lamS holds the warm-start
// band multipliers on entry and the solution on exit.  Block-wide: every thread calls it with identical arguments.
template <bool LOTS, class Src>
__device__ __noinline__ void prox_rootfind(const ProxArgs& p, const Src& src, int a, double b, double tau, double Delta,
                                              const ProxShared& sh, RootState& rs) {
  const int tid = threadIdx.x;
  const int G = rs.nobands ? 0 : p.G;
  double* scratch = sh.scratch;
  double* lamS = sh.lamS;
  double alpha = rs.alpha, beta = rs.beta;
  int amode = rs.amode;
  double a_min = -INFINITY, a_max = INFINITY, b_min = -INFINITY, b_max = INFINITY;   // brackets, computed lazily
  bool have_br = false;
  double P = 0, R = 0, sP = 0, sR = 0, Pa = 0, Ra = 0, pa = 0, ra = 0;
  int n_eval = 0;

  // range of the breakpoints in threshold space (only when a root find needs bisection)
  auto brackets = [&]() {
    double out[4];
    prox_brackets<LOTS>(src, Delta, scratch, out);
    a_min = out[0]; a_max = out[1]; b_min = out[2]; b_max = out[3];
    const double span = fmax(fmax(fabs(a_min), fabs(a_max)), fmax(fabs(b_min), fabs(b_max)));
    const double pad = 1e-9 * fmax(span, 1e-300) + 1e-300;
    if (!(a_min <= a_max)) { a_min = -1.0; a_max = 1.0; }
    if (!(b_min <= b_max)) { b_min = -1.0; b_max = 1.0; }
    a_min -= pad; a_max += pad; b_min -= pad; b_max += pad;
    have_br = true;
  };
  double Pb = 0, Rb = 0, pb2 = 0, rb2 = 0;     // sums of a second selected group (joint Newton)
  auto eval2 = [&](double al, double be, int s1, int s2) {
    ++n_eval;
    double out[12];
    prox_eval<LOTS>(src, lamS, G, al, be - Delta, s1, s2, scratch, out);
    P = out[0]; R = out[1]; sP = out[2]; sR = out[3];
    if (s1 >= 0 || s2 >= 0) { Pa = out[4]; Ra = out[5]; pa = out[6]; ra = out[7]; Pb = out[8]; Rb = out[9]; pb2 = out[10]; rb2 = out[11]; }
  };
  auto eval = [&](double al, double be, int sel) { eval2(al, be, sel, -1); };
  const double tol = 2e-15 * fmax(1.0, fabs(b) + (isfinite(tau) ? tau : 0.0));
  const double Pt = 0.5 * (tau + b), Rt = 0.5 * (tau - b);

  // (alpha, beta) for the current group multipliers; leaves the sums of the final thresholds (and of group sel)
  // section pass for the roots that asked for one (amode 1: ra on P(alpha), rb on R(beta); amode 0: rn on P - R)
  auto section = [&](Root1D* ra_, Root1D* rb_, Root1D* rn) {
    double fP[PROX_KSEC], fR[PROX_KSEC];
    ++n_eval;
    if (rn) {
      const double dx = (rn->hi - rn->lo) / (PROX_KSEC + 1), x0 = rn->lo + dx;
      prox_eval_multi<LOTS>(src, lamS, G, x0, dx, x0 - Delta, dx, scratch, fP, fR);
      for (int k = 0; k < PROX_KSEC; ++k) fP[k] -= fR[k];
      root_place(*rn, fP, x0, dx, b, -1);
      return;
    }
    const double dxa = ra_->sect ? (ra_->hi - ra_->lo) / (PROX_KSEC + 1) : 0.0, xa = ra_->sect ? ra_->lo + dxa : ra_->x;
    const double dxb = rb_->sect ? (rb_->hi - rb_->lo) / (PROX_KSEC + 1) : 0.0, xb = rb_->sect ? rb_->lo + dxb : rb_->x;
    prox_eval_multi<LOTS>(src, lamS, G, xa, dxa, xb - Delta, dxb, scratch, fP, fR);
    if (ra_->sect) root_place(*ra_, fP, xa, dxa, Pt, -1);
    if (rb_->sect) root_place(*rb_, fR, xb, dxb, Rt, +1);
  };
  // (alpha, beta) for the current group multipliers; leaves the sums of the final thresholds (and of group sel)
  auto solve_ab = [&](int sel) {
    double lmin = 0.0, lmax = 0.0;
    for (int g = 0; g < G; ++g) { lmin = fmin(lmin, lamS[g]); lmax = fmax(lmax, lamS[g]); }
    for (int attempt = 0; attempt < 4 && n_eval <= PROX_EVAL_CAP; ++attempt) {
      const double alo = a_min - lmax, ahi = a_max - lmin, blo = b_min - lmax, bhi = b_max - lmin;
      bool need = false;
      if (amode == 1) {
        Root1D ra_ = {fmin(fmax(alpha, alo), ahi), alo, ahi, 0, 0};
        Root1D rb_ = {fmin(fmax(beta, blo), bhi), blo, bhi, 0, 0};
        eval(ra_.x, rb_.x, sel);
        for (int it = 0; it < 80; ++it) {
          need = root_step(ra_, P, sP, Pt, -1, tol) | root_step(rb_, R, sR, Rt, +1, tol);
          if (need || (ra_.done && rb_.done)) break;
          if (n_eval > PROX_EVAL_CAP) break;
          if (ra_.sect || rb_.sect) section(&ra_, &rb_, nullptr);
          eval(ra_.x, rb_.x, sel);
        }
        alpha = ra_.x; beta = rb_.x;
        if (need) { brackets(); continue; }
        if (alpha >= beta) break;
        amode = 0; alpha = beta = 0.5 * (alpha + beta);
      } else {
        const double lo_b = fmin(alo, blo), hi_b = fmax(ahi, bhi);
        Root1D rn = {fmin(fmax(alpha, lo_b), hi_b), lo_b, hi_b, 0, 0};
        eval(rn.x, rn.x, sel);
        for (int it = 0; it < 80; ++it) {
          need = root_step(rn, P - R, sP + sR, b, -1, tol);
          if (need || rn.done) break;
          if (n_eval > PROX_EVAL_CAP) break;
          if (rn.sect) section(nullptr, nullptr, &rn);
          eval(rn.x, rn.x, sel);
        }
        alpha = beta = rn.x;
        if (need) { brackets(); continue; }
        if (!isfinite(tau) || P + R <= tau + tol) break;
        amode = 1;
      }
    }
  };

  // Fast path when one or two bands were active at the previous iteration: semismooth Newton on (alpha, beta,
  // lambda_g1[, lambda_g2]) jointly, one pass per step (the system is piecewise linear; from the warm start it lands
  // on the final piece in a few steps).  Anything unexpected falls through to the robust nested solve below.
  if (G > 0) {
    int g1 = -1, g2 = -1, nact = 0;
    for (int g = 0; g < G; ++g) if (lamS[g] != 0.0) { if (nact == 0) g1 = g; else if (nact == 1) g2 = g; ++nact; }
    if (nact >= 1 && nact <= 2) {
      const double bnd1 = lamS[g1] > 0.0 ? sh.band_hi[g1] : sh.band_lo[g1];
      const double bnd2 = g2 >= 0 ? (lamS[g2] > 0.0 ? sh.band_hi[g2] : sh.band_lo[g2]) : 0.0;
      const double gw1 = sh.gw0[g1], gw2 = g2 >= 0 ? sh.gw0[g2] : 0.0;
      const double sg1 = lamS[g1] > 0.0 ? 1.0 : -1.0, sg2 = g2 >= 0 ? (lamS[g2] > 0.0 ? 1.0 : -1.0) : 1.0;
      const double l1_0 = lamS[g1], l2_0 = g2 >= 0 ? lamS[g2] : 0.0;
      double al = alpha, be = beta, l1 = l1_0, l2 = l2_0;
      bool ok = false;
      for (int it = 0; it < 10; ++it) {
        eval2(al, be, g1, g2);
        const double F1 = gw1 + Pa - Ra - bnd1, F2 = g2 >= 0 ? gw2 + Pb - Rb - bnd2 : 0.0;
        double FA, FB;                                   // residuals of the (alpha, beta) equations
        if (amode == 1) { FA = P - Pt; FB = R - Rt; } else { FA = P - R - b; FB = 0.0; }
        if (fabs(F1) <= tol && fabs(F2) <= tol && fabs(FA) <= tol && fabs(FB) <= tol) { ok = true; break; }
        // reduced Newton system in (dl1, dl2)
        double M11, M12, M22, r1, r2;
        const double s1 = pa + ra, s2 = pb2 + rb2;
        if (amode == 1) {
          if (!(sP > 0.0) || !(sR > 0.0)) break;
          M11 = -s1 + pa * pa / sP + ra * ra / sR; M22 = -s2 + pb2 * pb2 / sP + rb2 * rb2 / sR;
          M12 = pa * pb2 / sP + ra * rb2 / sR;
          r1 = -F1 + pa * FA / sP - ra * FB / sR; r2 = -F2 + pb2 * FA / sP - rb2 * FB / sR;
        } else {
          const double st = sP + sR;
          if (!(st > 0.0)) break;
          M11 = -s1 + s1 * s1 / st; M22 = -s2 + s2 * s2 / st; M12 = s1 * s2 / st;
          r1 = -F1 + s1 * FA / st; r2 = -F2 + s2 * FA / st;
        }
        double d1, d2 = 0.0;
        if (g2 >= 0) {
          const double det = M11 * M22 - M12 * M12;
          if (!(fabs(det) > 1e-300)) break;
          d1 = (r1 * M22 - M12 * r2) / det; d2 = (M11 * r2 - M12 * r1) / det;
        } else {
          if (!(fabs(M11) > 1e-300)) break;
          d1 = r1 / M11;
        }
        if (amode == 1) { al += (FA - pa * d1 - pb2 * d2) / sP; be += (-FB - ra * d1 - rb2 * d2) / sR; }
        else { al += (FA - s1 * d1 - s2 * d2) / (sP + sR); be = al; }
        l1 += d1; l2 += d2;
        if (!(l1 == l1) || !(l2 == l2) || !(al == al) || !(be == be)) break;
        __syncthreads();
        if (tid == 0) { lamS[g1] = l1; if (g2 >= 0) lamS[g2] = l2; }
        __syncthreads();
      }
      // accept only a consistent solution: multiplier signs kept, theta >= 0 / cap slack; otherwise restore and fall through
      bool good = ok && l1 * sg1 > 0.0 && (g2 < 0 || l2 * sg2 > 0.0);
      if (good) good = amode == 1 ? (al >= be) : (!isfinite(tau) || P + R <= tau + tol);
      __syncthreads();
      if (good) { alpha = al; beta = be; }
      else if (tid == 0) { lamS[g1] = l1_0; if (g2 >= 0) lamS[g2] = l2_0; }
      __syncthreads();
    }
  }

  bool gs_done = false;      // every band holds (or there are none)
  for (int round = 0; round < rs.max_rounds && n_eval <= PROX_EVAL_CAP; ++round) {
    solve_ab(-1);
    if (G == 0) { gs_done = true; break; }
    // all group sums at the current solution (deterministic binned pass)
    prox_group_sums<LOTS>(src, lamS, G, alpha, beta - Delta, sh.gw0, sh.gbin, sh.gsum);
    if (tid == 0) {
      int sel = -1, sgn = 0; double worst = 8.0 * tol;
      for (int g = 0; g < G; ++g) {
        const double bl_ = sh.band_lo[g], bh_ = sh.band_hi[g];
        double viol; int sg;
        if (lamS[g] > 0.0) { viol = fabs(sh.gsum[g] - bh_); sg = +1; }
        else if (lamS[g] < 0.0) { viol = fabs(sh.gsum[g] - bl_); sg = -1; }
        else if (sh.gsum[g] > bh_) { viol = sh.gsum[g] - bh_; sg = +1; }
        else { viol = bl_ - sh.gsum[g]; sg = -1; }
        if (viol > worst) { worst = viol; sel = g; sgn = sg; }
      }
      // past the usual 2G+2 rounds (a caller that allows more) the rounds stop at rounding level: with several active bands
      // the sums carry ~1e-14 of rounding noise and two bands can hand a violation of that size back and forth for ever
      if (sel >= 0 && round >= 2 * G + 2 && worst <= 512.0 * tol) sel = -1;
      sh.selS[0] = sel; sh.selS[1] = sgn;
    }
    __syncthreads();
    const int sel = sh.selS[0], sgn = sh.selS[1];
    if (sel < 0) { gs_done = true; break; }
    // scalar problem in m = sgn * lambda_sel >= 0:  h(m) = sgn * (S_sel - bound) is non-increasing, want h = 0 or m = 0
    if (!have_br) brackets();
    const double Lmax = 2.0 * (fmax(a_max, b_max) - fmin(a_min, b_min)) + 1.0;
    const double bound = sgn > 0 ? sh.band_hi[sel] : sh.band_lo[sel];
    const double gw = sh.gw0[sel];
    double m = sgn * lamS[sel], mlo = 0.0, mhi = Lmax;
    bool lo_known = false;      // h(mlo) > 0 established
    for (int it = 0; it < 60 && n_eval <= PROX_EVAL_CAP; ++it) {
      __syncthreads();
      if (tid == 0) lamS[sel] = sgn * m;
      __syncthreads();
      solve_ab(sel);
      const double h = sgn * (gw + Pa - Ra - bound);
      if (fabs(h) <= tol) break;
      if (m == 0.0 && h < 0.0) break;                    // band inactive at lambda = 0
      double slope = pa + ra;
      if (amode == 1) slope -= (sP > 0.0 ? pa * pa / sP : 0.0) + (sR > 0.0 ? ra * ra / sR : 0.0);
      else slope -= (sP + sR > 0.0 ? (pa + ra) * (pa + ra) / (sP + sR) : 0.0);
      if (h > 0.0) { mlo = m; lo_known = true; } else mhi = m;
      double mn = slope > 1e-300 ? m + h / slope : NAN;
      if (!(mn == mn)) mn = lo_known || mlo > 0.0 ? 0.5 * (mlo + mhi) : 0.0;
      if (mn <= mlo) mn = lo_known ? 0.5 * (mlo + mhi) : 0.0;
      if (mn >= mhi) mn = 0.5 * (mlo + mhi);
      if (mn == m) break;
      m = mn;
    }
  }
  __syncthreads();
  rs.alpha = alpha; rs.beta = beta; rs.amode = amode; rs.n_eval += n_eval;
  if (n_eval > PROX_EVAL_CAP) rs.capped = 1;
  else if (!gs_done) rs.capped = 2;
}

__device__ __forceinline__ double next_window(const ProxArgs& p, double alpha, double beta, double mv) {
  return fmax(p.win_mult * mv, 1e-9 + 1e-7 * (fabs(alpha) + fabs(beta)));
}

// ------------------------------------------------------------------------------------------------ slow path
// Whole z-update of one account from a source that can enumerate every asset: root find (windowed for SrcSmem),
// residual check, convergence mask, rho adaptation, output / returned weights.
template <bool LOTS, class Src>
__device__ __forceinline__ void prox_body(const ProxArgs& p, int mode, Src& src, int a, double gam, double c,
                                          double kappa, double lam_b, const ProxShared& sh0, bool windowed) {
  const int tid = threadIdx.x, nt = blockDim.x;
  ProxShared sh = sh0;
  sh.band_lo = p.band_lo + (int64_t)a * p.G; sh.band_hi = p.band_hi + (int64_t)a * p.G; sh.gw0 = p.gw0 + (int64_t)a * p.G;
  double* lamS = sh.lamS;
  double cg = c * gam;
  const double Delta = lam_b + kappa;
  const double tau = p.tau ? p.tau[a] : INFINITY;
  const double b = p.ap.bsum[a];
  const int G = p.G;
  for (int g = tid; g < G; g += nt) lamS[g] = p.lamG[(int64_t)a * G + g];
  __syncthreads();

  RootState rs;
  rs.alpha = p.ap.alpha[a]; rs.beta = p.ap.beta[a]; rs.amode = p.ap.mode[a]; rs.n_eval = 0; rs.nobands = 0; rs.capped = 0;
  rs.max_rounds = 1 << 30;       // this form has no joint Newton iteration to polish with: rounds until every band holds
  if (!(rs.amode == 1 && isfinite(tau))) { rs.amode = 0; rs.beta = rs.alpha; }
  const double alpha_w = rs.alpha, beta_w = rs.beta;       // warm start (previous iteration's thresholds)
  const int amode_w = rs.amode;
  const double* lam_w = p.lamG + (int64_t)a * G;
  src.classify(alpha_w, beta_w, lam_w, windowed ? p.ap.win[a] : INFINITY, (int*)sh.scratch);
  for (int wpass = 0; wpass < 2; ++wpass) {
    prox_rootfind<LOTS>(p, src, a, b, tau, Delta, sh, rs);
    if (src.window_ok(rs.alpha, rs.beta, lamS)) break;
    // the solution left the window the live list was built for: rebuild it with every asset and solve again
    rs.alpha = alpha_w; rs.beta = beta_w; rs.amode = amode_w; rs.capped = 0;
    __syncthreads();
    for (int g = tid; g < G; g += nt) lamS[g] = lam_w[g];
    __syncthreads();
    src.classify(alpha_w, beta_w, lam_w, INFINITY, (int*)sh.scratch);
  }
  __syncthreads();
  const double alpha = rs.alpha, beta = rs.beta;

  // ---------------------------------------------------------------- check: residuals, mask, rho adaptation
  double c_new = c;
  int finished = 0;
  const double bdf = beta - Delta;
  if (mode & PROX_CHECK) {
    double rr[3];
    prox_check<LOTS>(p, src, lamS, a, alpha, bdf, lam_b, cg, sh.scratch, rr);
    const double rp = rr[0], rd = rr[1];
    const bool bad = !(rp < INFINITY) || !(rd < INFINITY);
    const bool conv = !bad && rr[2] > 0.0 && !rs.capped;      // never certify on an unfinished root find
    if (tid == 0) {
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_PRIMAL] = rp;
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_DUAL] = rd;
    }
    if (conv || bad) {
      finished = 1;
      if (tid == 0) p.ap.conv[a] = bad ? -1 : 1;
    } else if (p.adapt && p.iter >= p.adapt_start && p.iter - p.ap.nadapt[a] >= p.adapt_every) {
      // H7: only accounts that are unusually slow are re-scaled (typical accounts finish before PRISM_ADAPT_START);
      // rho <- rho sqrt(r_p / r_d), clipped, applied when the two scaled residuals are out of balance
      const double ratio = sqrt(rp / fmax(rd, 1e-300));
      if (ratio > 3.0 || ratio < 1.0 / 3.0) {
        c_new = c * fmin(fmax(ratio, 0.2), 5.0);
        if (tid == 0) { p.ap.c[a] = c_new; p.ap.refactor[a] = 1; }
      }
      if (tid == 0) p.ap.nadapt[a] = p.iter;
    }
  }
  if (mode & PROX_FINAL) finished = 1;

  // ---------------------------------------------------------------- output pass (e.T, e.ir refer to the old rho)
  prox_output<LOTS>(p, src, lamS, a, alpha, bdf, lam_b, gam, c, c_new, finished);
  double mv_l = 0.0;
  for (int g = 0; g < G; ++g) mv_l = fmax(mv_l, fabs(lamS[g] - lam_w[g]));
  __syncthreads();
  for (int g = tid; g < G; g += nt) p.lamG[(int64_t)a * G + g] = lamS[g];
  if (tid == 0) {
    p.ap.alpha[a] = alpha; p.ap.beta[a] = beta; p.ap.mode[a] = rs.amode;
    // next window: a multiple of how far the thresholds moved in this launch
    p.ap.win[a] = next_window(p, alpha, beta, fmax(fmax(fabs(alpha - alpha_w), fabs(beta - beta_w)), mv_l));
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
  __syncthreads();
}

