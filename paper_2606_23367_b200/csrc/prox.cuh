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
  double eps;
  int32_t adapt, iter;
};

enum { PROX_CHECK = 1, PROX_FINAL = 2, PROX_INIT = 4 };
#define PRISM_ADAPT_START 200   // first iteration at which an account's rho may be adapted
#define PRISM_ADAPT_EVERY 100   // minimum iterations between two adaptations of one account

struct ElemConst {        // per-element quantities that do not depend on the trial thresholds
  double u, ir, bl, bh, sl, sh, w0;     // u = v - w0, ir = 1 / rho_i, buy range [bl, bh], sell range [sl, sh]
};

__device__ __forceinline__ void elem_ranges(ElemConst& e, double lo, double hi) {
  e.bl = fmax(lo - e.w0, 0.0);
  e.bh = fmax(hi - e.w0, 0.0);
  e.sl = fmax(e.w0 - hi, 0.0);
  e.sh = fmax(e.w0 - lo, 0.0);
}

// buy amount at threshold a = alpha + lambda_g; mv = 1/rho_i if strictly inside its range (|slope| of the piece)
__device__ __forceinline__ double buy_amt(const ElemConst& e, double lam_b, double a, double& mv) {
  const double raw = e.u - (lam_b + a) * e.ir;
  mv = (raw > e.bl && raw < e.bh) ? e.ir : 0.0;
  return fmin(fmax(raw, e.bl), e.bh);
}

template <bool LOTS>
__device__ __forceinline__ double sell_amt(const ElemConst& e, double kappa, double bt, const double* slope,
                                           const double* width, int nl, double& mv) {
  double raw, inside = 0.0;
  double sh = e.sh;
  if (LOTS && nl > 0) {
    raw = 0.0;
    double Q = 0.0;
    for (int l = 0; l < nl; ++l) {
      const double r = (bt - kappa - slope[l]) * e.ir - e.u - Q;
      const double ql = width[l];
      if (r > 0.0 && r < ql) inside = 1.0;
      raw += fmin(fmax(r, 0.0), ql);
      Q += ql;
    }
    sh = fmin(sh, Q);
  } else {
    raw = (bt - kappa) * e.ir - e.u;
    inside = 1.0;
  }
  mv = (inside > 0.0 && raw > e.sl && raw < sh) ? e.ir : 0.0;
  return fmin(fmax(raw, e.sl), sh);
}

// One bracketed Newton step on a continuous piecewise-linear monotone function.
// dir = +1: g increasing in x, -1: decreasing.  slope = |g'| at x (0 on a flat piece).
struct Root1D {
  double x, lo, hi;
  int done;
};
__device__ __forceinline__ void root_step(Root1D& r, double g, double slope, double target, int dir, double tol) {
  if (r.done) return;
  const double diff = g - target;
  if (fabs(diff) <= tol) { r.done = 1; return; }
  const bool too_big = (dir > 0) ? (diff > 0.0) : (diff < 0.0);   // x lies right of the root
  if (too_big) r.hi = r.x; else r.lo = r.x;
  double xn = (slope > 0.0) ? r.x - (double)dir * diff / slope : NAN;
  if (!(xn > r.lo && xn < r.hi)) xn = 0.5 * (r.lo + r.hi);
  if (xn == r.x || !(r.hi - r.lo > 0.0) || !(xn > r.lo && xn < r.hi)) { r.done = 1; r.x = (xn == xn) ? xn : r.x; return; }
  r.x = xn;
}

// ---------------------------------------------------------------------------------------------- element sources
// Generic source: every pass re-reads the account from global memory (any N, lots, per-asset caps).
template <bool LOTS>
struct SrcGlobal {
  const ProxArgs& p;
  int64_t row, rowp;
  double icg, lo_a, hi_a;
  __device__ SrcGlobal(const ProxArgs& p_, int a, double cg, double lo, double hi)
      : p(p_), row((int64_t)a * p_.N), rowp((int64_t)a * p_.ldw), icg(1.0 / cg), lo_a(lo), hi_a(hi) {}
  __device__ __forceinline__ void set_scale(double cg) { icg = 1.0 / cg; }
  __device__ __forceinline__ void load(int64_t i, ElemConst& e, int& g, int& nl, const double*& sl, const double*& wd) const {
    const int64_t idx = row + i;
    e.w0 = p.w0[idx];
    e.u = p.v[rowp + i] - e.w0;
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
  __device__ __forceinline__ void store_v(int64_t i, double vv) const { p.v[rowp + i] = vv; }
};

// Shared-memory source: u = v - w0 and w0 of the whole account stay in shared memory for the kernel (2 x 8 B x N),
// so a trial evaluation touches no HBM: only 1/d_i, the exclusion byte and the group id (shared by many CTAs or
// tiny; L1/L2 resident).  Each thread reads back only what it wrote: no barrier needed.  No lots, no per-asset caps.
struct SrcSmem {
  const ProxArgs& p;
  int64_t row, rowp;
  double icg, lo_a, hi_a;
  double *us, *ws;
  __device__ SrcSmem(const ProxArgs& p_, int a, double cg, double lo, double hi, double* smem)
      : p(p_), row((int64_t)a * p_.N), rowp((int64_t)a * p_.ldw), icg(1.0 / cg), lo_a(lo), hi_a(hi), us(smem), ws(smem + p_.N) {
    for (int64_t i = threadIdx.x; i < p.N; i += blockDim.x) {
      const double w = p.w0[row + i];
      ws[i] = w;
      us[i] = p.v[rowp + i] - w;
    }
  }
  __device__ __forceinline__ void load(int64_t i, ElemConst& e, int& g) const {
    e.w0 = ws[i]; e.u = us[i];
    e.ir = p.invd[i] * icg;
    const bool ex = p.excl && p.excl[row + i];
    elem_ranges(e, ex ? 0.0 : lo_a, ex ? 0.0 : hi_a);
    g = p.G ? p.group_id[i] : 0;
  }
  template <class F>
  __device__ __forceinline__ void for_each(F f) const {
    for (int64_t i = threadIdx.x; i < p.N; i += blockDim.x) {
      ElemConst e; int g;
      load(i, e, g);
      f(i, e, g, 0, (const double*)nullptr, (const double*)nullptr);
    }
  }
  template <class F>
  __device__ __forceinline__ void for_each_uniform(F f) const {
    for (int64_t i0 = 0; i0 < p.N; i0 += blockDim.x) {
      const int64_t i = i0 + threadIdx.x;
      const bool valid = i < p.N;
      ElemConst e; int g = 0;
      if (valid) load(i, e, g);
      f(valid, i, e, g, 0, (const double*)nullptr, (const double*)nullptr);
    }
  }
  __device__ __forceinline__ void store_v(int64_t i, double vv) const { p.v[rowp + i] = vv; }
};

template <bool LOTS, class Src>
__device__ __forceinline__ void prox_body(const ProxArgs& p, int mode, Src& src, int a, double gam, double c) {
  __shared__ double scratch[8 * 32];
  __shared__ double gbin[16 * PRISM_MAX_GROUPS];    // per-warp group bins (deterministic accumulation)
  __shared__ double lamS[PRISM_MAX_GROUPS];
  __shared__ double gsum[PRISM_MAX_GROUPS];
  __shared__ int selS[2];
  const int tid = threadIdx.x, nt = blockDim.x;
  const int64_t N = p.N, row = (int64_t)a * N, rowp = (int64_t)a * p.ldw;
  double cg = c * gam;
  const double kappa = p.kappa ? p.kappa[a] : 0.0;
  const double lam_b = kappa + (p.c_buy ? p.c_buy[a] : 0.0);
  const double tau = p.tau ? p.tau[a] : INFINITY;
  const double b = p.ap.bsum[a];
  const int G = p.G;
  for (int g = tid; g < G; g += nt) lamS[g] = p.lamG[(int64_t)a * G + g];
  __syncthreads();

  double alpha = p.ap.alpha[a], beta = p.ap.beta[a];
  int amode = p.ap.mode[a];
  if (!(amode == 1 && isfinite(tau))) { amode = 0; beta = alpha; }
  double a_min, a_max, b_min, b_max;
  double P = 0, R = 0, sP = 0, sR = 0, Pa = 0, Ra = 0, pa = 0, ra = 0;

  // pass 0: totals at the warm start and the range of the breakpoints (brackets)
  {
    double lP = 0, lR = 0, lsP = 0, lsR = 0, x4 = INFINITY, x5 = -INFINITY, x6 = INFINITY, x7 = -INFINITY;
    src.for_each([&](int64_t, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
      double mvb, mvs;
      const double lg = G ? lamS[g] : 0.0;
      lP += buy_amt(e, lam_b, alpha + lg, mvb);
      lR += sell_amt<LOTS>(e, kappa, beta + lg, sl, wd, nl, mvs);
      lsP += mvb; lsR += mvs;
      const double rho = 1.0 / e.ir;
      if (e.bh > e.bl) { x4 = fmin(x4, rho * (e.u - e.bh) - lam_b); x5 = fmax(x5, rho * (e.u - e.bl) - lam_b); }
      double sh = e.sh, s_first = 0.0, s_last = 0.0;
      if (LOTS && nl > 0) { double Q = 0; for (int l = 0; l < nl; ++l) Q += wd[l]; sh = fmin(sh, Q); s_first = sl[0]; s_last = sl[nl - 1]; }
      if (sh > e.sl) { x6 = fmin(x6, rho * (e.u + e.sl) + kappa + s_first); x7 = fmax(x7, rho * (e.u + sh) + kappa + s_last); }
    });
    double val[8] = {lP, lR, lsP, lsR, x4, x5, x6, x7};
    const int op[8] = {0, 0, 0, 0, 2, 1, 2, 1};
    block_reduce<8>(val, op, scratch);
    P = val[0]; R = val[1]; sP = val[2]; sR = val[3];
    a_min = val[4]; a_max = val[5]; b_min = val[6]; b_max = val[7];
  }
  // one pass: totals at thresholds (al, be) shifted by the group multipliers; with sel >= 0 also the sums of group sel
  int n_eval = 1;
  auto eval = [&](double al, double be, int sel) {
    ++n_eval;
    double lP = 0, lR = 0, lsP = 0, lsR = 0, x4 = 0, x5 = 0, x6 = 0, x7 = 0;
    src.for_each([&](int64_t, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
      double mvb, mvs;
      const double lg = G ? lamS[g] : 0.0;
      const double pb = buy_amt(e, lam_b, al + lg, mvb);
      const double ps = sell_amt<LOTS>(e, kappa, be + lg, sl, wd, nl, mvs);
      lP += pb; lR += ps; lsP += mvb; lsR += mvs;
      if (g == sel) { x4 += pb; x5 += ps; x6 += mvb; x7 += mvs; }
    });
    if (sel >= 0) {
      double val[8] = {lP, lR, lsP, lsR, x4, x5, x6, x7};
      const int op[8] = {0, 0, 0, 0, 0, 0, 0, 0};
      block_reduce<8>(val, op, scratch);
      P = val[0]; R = val[1]; sP = val[2]; sR = val[3]; Pa = val[4]; Ra = val[5]; pa = val[6]; ra = val[7];
    } else {
      double val[4] = {lP, lR, lsP, lsR};
      const int op[4] = {0, 0, 0, 0};
      block_reduce<4>(val, op, scratch);
      P = val[0]; R = val[1]; sP = val[2]; sR = val[3];
    }
  };
  const double span = fmax(fmax(fabs(a_min), fabs(a_max)), fmax(fabs(b_min), fabs(b_max)));
  const double pad = 1e-9 * fmax(span, 1e-300) + 1e-300;
  if (!(a_min <= a_max)) { a_min = -1.0; a_max = 1.0; }
  if (!(b_min <= b_max)) { b_min = -1.0; b_max = 1.0; }
  a_min -= pad; a_max += pad; b_min -= pad; b_max += pad;
  const double tol = 2e-15 * fmax(1.0, fabs(b) + (isfinite(tau) ? tau : 0.0));
  const double Pt = 0.5 * (tau + b), Rt = 0.5 * (tau - b);
  const double Lmax = 2.0 * (fmax(a_max, b_max) - fmin(a_min, b_min)) + 1.0;
  bool fresh = true;     // P, R, ... correspond to (alpha, beta, lamS, sel = -1)

  // (alpha, beta) for the current group multipliers; leaves the sums of the final thresholds (and of group sel)
  auto solve_ab = [&](int sel) {
    double lmin = 0.0, lmax = 0.0;
    for (int g = 0; g < G; ++g) { lmin = fmin(lmin, lamS[g]); lmax = fmax(lmax, lamS[g]); }
    const double alo = a_min - lmax, ahi = a_max - lmin, blo = b_min - lmax, bhi = b_max - lmin;
    for (int attempt = 0; attempt < 3; ++attempt) {
      if (amode == 1) {
        Root1D ra_ = {fmin(fmax(alpha, alo), ahi), alo, ahi, 0};
        Root1D rb_ = {fmin(fmax(beta, blo), bhi), blo, bhi, 0};
        if (!fresh || sel >= 0 || ra_.x != alpha || rb_.x != beta) eval(ra_.x, rb_.x, sel);
        fresh = false;
        for (int it = 0; it < 80; ++it) {
          root_step(ra_, P, sP, Pt, -1, tol);
          root_step(rb_, R, sR, Rt, +1, tol);
          if (ra_.done && rb_.done) break;
          eval(ra_.x, rb_.x, sel);
        }
        alpha = ra_.x; beta = rb_.x;
        if (alpha >= beta) break;
        amode = 0; alpha = beta = 0.5 * (alpha + beta);
      } else {
        const double lo_b = fmin(alo, blo), hi_b = fmax(ahi, bhi);
        Root1D rn = {fmin(fmax(alpha, lo_b), hi_b), lo_b, hi_b, 0};
        if (!fresh || sel >= 0 || rn.x != alpha || beta != alpha) eval(rn.x, rn.x, sel);
        fresh = false;
        for (int it = 0; it < 80; ++it) {
          root_step(rn, P - R, sP + sR, b, -1, tol);
          if (rn.done) break;
          eval(rn.x, rn.x, sel);
        }
        alpha = beta = rn.x;
        if (!isfinite(tau) || P + R <= tau + tol) break;
        amode = 1;
      }
    }
  };

  for (int round = 0; round < 2 * G + 2; ++round) {
    solve_ab(-1);
    if (G == 0) break;
    // all group sums at the current solution (deterministic binned pass)
    for (int g = tid; g < 16 * G; g += nt) gbin[g] = 0.0;
    __syncthreads();
    src.for_each_uniform([&](bool valid, int64_t, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
      double t = 0.0;
      if (valid) {
        double mvb, mvs;
        t = buy_amt(e, lam_b, alpha + lamS[g], mvb) - sell_amt<LOTS>(e, kappa, beta + lamS[g], sl, wd, nl, mvs);
      }
      warp_group_add(gbin, G, valid ? g : 0, t, valid);
    });
    __syncthreads();
    for (int g = tid; g < G; g += nt) gsum[g] = p.gw0[(int64_t)a * G + g] + group_total(gbin, G, g);
    __syncthreads();
    if (tid == 0) {
      int sel = -1, sgn = 0; double worst = 8.0 * tol;
      for (int g = 0; g < G; ++g) {
        const double bl_ = p.band_lo[(int64_t)a * G + g], bh_ = p.band_hi[(int64_t)a * G + g];
        double viol; int sg;
        if (lamS[g] > 0.0) { viol = fabs(gsum[g] - bh_); sg = +1; }
        else if (lamS[g] < 0.0) { viol = fabs(gsum[g] - bl_); sg = -1; }
        else if (gsum[g] > bh_) { viol = gsum[g] - bh_; sg = +1; }
        else { viol = bl_ - gsum[g]; sg = -1; }
        if (viol > worst) { worst = viol; sel = g; sgn = sg; }
      }
      selS[0] = sel; selS[1] = sgn;
    }
    __syncthreads();
    const int sel = selS[0], sgn = selS[1];
    if (sel < 0) break;
    // scalar problem in m = sgn * lambda_sel >= 0:  h(m) = sgn * (S_sel - bound) is non-increasing, want h = 0 or m = 0
    const double bound = sgn > 0 ? p.band_hi[(int64_t)a * G + sel] : p.band_lo[(int64_t)a * G + sel];
    const double gw = p.gw0[(int64_t)a * G + sel];
    double m = sgn * lamS[sel], mlo = 0.0, mhi = Lmax;
    bool lo_known = false;      // h(mlo) > 0 established
    for (int it = 0; it < 60; ++it) {
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
    fresh = false;
  }
  __syncthreads();

  // ---------------------------------------------------------------- check: residuals, mask, rho adaptation
  double rescale = 1.0;
  int finished = 0;
  if (mode & PROX_CHECK) {
    double nx = 0, nz = 0, nrp = 0, nrd = 0, nPx = 0, ny = 0, nq = 0;
    src.for_each([&](int64_t i, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
      double mvb, mvs;
      const double lg = G ? lamS[g] : 0.0;
      const double tr = buy_amt(e, lam_b, alpha + lg, mvb) - sell_amt<LOTS>(e, kappa, beta + lg, sl, wd, nl, mvs);
      const double z = e.w0 + tr;
      const double y = (e.u - tr) / e.ir;                 // rho (v - z)
      const double x = p.xs[rowp + i], pq = p.pxq[rowp + i];
      const double qi = p.q ? p.q[rowp + i] : -p.mu[row + i];
      nx = fmax(nx, fabs(x)); nz = fmax(nz, fabs(z)); nrp = fmax(nrp, fabs(x - z));
      nrd = fmax(nrd, fabs(pq + y)); nPx = fmax(nPx, fabs(pq - qi)); ny = fmax(ny, fabs(y)); nq = fmax(nq, fabs(qi));
      if (!(z == z) || !(x == x) || !(e.u == e.u)) nrp = INFINITY;     // fmax drops NaN: poison explicitly
    });
    double val[7] = {nx, nz, nrp, nrd, nPx, ny, nq};
    const int op[7] = {1, 1, 1, 1, 1, 1, 1};
    block_reduce<7>(val, op, scratch);
    const double rp = val[2] / fmax(fmax(val[0], val[1]), 1e-300);
    const double rd = val[3] / fmax(fmax(val[4], fmax(val[5], val[6])), 1e-300);
    const bool bad = !(rp < INFINITY) || !(rd < INFINITY);
    const bool conv = !bad && rp <= p.eps && rd <= p.eps;
    if (tid == 0) {
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_PRIMAL] = rp;
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_DUAL] = rd;
    }
    if (conv || bad) {
      finished = 1;
      if (tid == 0) p.ap.conv[a] = bad ? -1 : 1;
    } else if (p.adapt && p.iter >= PRISM_ADAPT_START && p.iter - p.ap.nadapt[a] >= PRISM_ADAPT_EVERY) {
      // H7: only accounts that are unusually slow are re-scaled (typical accounts finish before PRISM_ADAPT_START);
      // rho <- rho sqrt(r_p / r_d), clipped, applied when the two scaled residuals are out of balance
      const double ratio = sqrt(rp / fmax(rd, 1e-300));
      if (ratio > 3.0 || ratio < 1.0 / 3.0) {
        const double cn = c * fmin(fmax(ratio, 0.2), 5.0);
        rescale = c / cn;          // v' = z + (rho/rho') (v - z) keeps y = rho (v - z) unchanged
        c = cn; cg = c * gam;
        if (tid == 0) { p.ap.c[a] = c; p.ap.refactor[a] = 1; }
      }
      if (tid == 0) p.ap.nadapt[a] = p.iter;
    }
  }
  if (mode & PROX_FINAL) finished = 1;

  // ---------------------------------------------------------------- output pass (e.ir still refers to the old rho)
  const double igc = 1.0 / (gam * (1.0 + c));
  src.for_each([&](int64_t i, const ElemConst& e, int g, int nl, const double* sl, const double* wd) {
    double mvb, mvs;
    const double lg = G ? lamS[g] : 0.0;
    const double tr = buy_amt(e, lam_b, alpha + lg, mvb) - sell_amt<LOTS>(e, kappa, beta + lg, sl, wd, nl, mvs);
    const double z = e.w0 + tr;
    if (finished) { p.w_out[row + i] = z; return; }
    const double y = (e.u - tr) / e.ir;                    // rho_old (v - z)
    if (rescale != 1.0) src.store_v(i, z + rescale * (e.u - tr));
    const double dinv = p.invd[i];
    const double rho = cg / dinv;                          // new rho_i
    const double qi = p.q ? p.q[rowp + i] : -p.mu[row + i];
    const double r = rho * z - y - qi;
    const double rt = r * dinv * igc;                      // M_i = gamma d_i (1 + c)
    p.rt[rowp + i] = rt;
    p.cc[rowp + i] = rt - z;
  });
  for (int g = tid; g < G; g += nt) p.lamG[(int64_t)a * G + g] = lamS[g];
  if (tid == 0) {
    p.resid[(int64_t)a * PRISM_NRES + PRISM_R_RESERVED] += (double)n_eval;   // trial evaluations (passes) so far
    p.ap.alpha[a] = alpha; p.ap.beta[a] = beta; p.ap.mode[a] = amode;
    if (finished) {
      p.ap.done[a] = 1;
      p.ap.iters[a] = p.iter;
      atomicAdd(&p.counters[0], 1);
      double* du = p.duals + (int64_t)a * PRISM_NDUAL(G);
      du[0] = 0.5 * (alpha + beta);
      du[1] = 0.5 * (alpha - beta);
      for (int g = 0; g < G; ++g) { du[2 + g] = fmax(lamS[g], 0.0); du[2 + G + g] = fmax(-lamS[g], 0.0); }
      p.resid[(int64_t)a * PRISM_NRES + PRISM_R_RHO] = c;
    }
  }
}

// generic kernel: any N, lots, per-asset caps
template <bool LOTS>
__global__ void __launch_bounds__(512) k_prox(ProxArgs p, int mode) {
  const int a = blockIdx.x;
  if (p.ap.done[a]) return;
  const double gam = p.gamma[a], c = p.ap.c[a];
  SrcGlobal<LOTS> src(p, a, c * gam, p.lo[a], p.hi[a]);
  prox_body<LOTS>(p, mode, src, a, gam, c);
}

// shared-memory-resident kernel: 16 N bytes of dynamic shared memory, no lots, no per-asset caps
__global__ void __launch_bounds__(512, 1) k_prox_smem(ProxArgs p, int mode) {
  extern __shared__ __align__(16) double prox_smem[];
  const int a = blockIdx.x;
  if (p.ap.done[a]) return;
  const double gam = p.gamma[a], c = p.ap.c[a];
  SrcSmem src(p, a, c * gam, p.lo[a], p.hi[a], prox_smem);
  prox_body<false>(p, mode, src, a, gam, c);
}
