// diag.cuh - external diagnostics of Section 4.4 for given weights (and multipliers), one CTA
// per account, and the status vocabulary of Table 14.  Depends only on the problem data, w,
// duals and gS = gamma Sigma (w - w_b) (computed by the fp64 Sigma-apply, H8); never on solver state.
#pragma once
#include "common.cuh"
#include "diag_args.cuh"

template <bool LOTS>
__global__ void __launch_bounds__(256) k_diag(DiagArgs p) {
  __shared__ double scratch[8 * 32];
  __shared__ double gbin[8 * PRISM_MAX_GROUPS];
  __shared__ double gsum[PRISM_MAX_GROUPS];
  __shared__ double lam[PRISM_MAX_GROUPS];
  const int a = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const int64_t N = p.N, row = (int64_t)a * N, rowp = (int64_t)a * p.ldw;
  const int G = p.G, L = PRISM_MAX_LOTS;
  const bool have = p.duals != nullptr;
  const double* du = have ? p.duals + (int64_t)a * PRISM_NDUAL(G) : nullptr;
  const double nu = have ? du[0] : 0.0, theta = have ? du[1] : 0.0;
  for (int g = tid; g < 8 * G; g += nt) gbin[g] = 0.0;
  for (int g = tid; g < G; g += nt) lam[g] = have ? du[2 + g] - du[2 + G + g] : 0.0;
  __syncthreads();
  const double lo_a = p.lo[a], hi_a = p.hi[a];
  const double kappa = p.kappa ? p.kappa[a] : 0.0, cb = p.c_buy ? p.c_buy[a] : 0.0;
  const double tau = p.tau ? p.tau[a] : INFINITY;
  const double lamt = kappa + theta, dl = p.delta;
  double sw = 0, rbox = 0, turn = 0, fobj = 0, rstat = 0;
  bool bad = false;
  for (int64_t i0 = 0; i0 < N; i0 += nt) {
    const int64_t i = i0 + tid;
    const bool valid = i < N;
    if (G) warp_group_add(gbin, G, valid ? p.group_id[i] : 0, valid ? p.w[row + i] : 0.0, valid);
    if (!valid) continue;
    const double w = p.w[row + i], w0 = p.w0[row + i], mu = p.mu[row + i];
    double lo = lo_a, hi = p.hi_full ? p.hi_full[row + i] : hi_a;
    if (p.excl && p.excl[row + i]) { lo = 0.0; hi = 0.0; }
    if (!(w == w) || isinf(w)) bad = true;
    const double dw = w - w0;
    sw += w;
    turn += fabs(dw);
    rbox = fmax(rbox, fmax(lo - w, w - hi));
    // objective f(w) (PAPER.md:109 in the SURVEY 8.0 form)
    const double x = p.w_b ? w - p.w_b[row + i] : w;
    const double gs = p.gS[rowp + i];
    double pen = kappa * fabs(dw) + cb * fmax(dw, 0.0);
    // subdifferential interval of phi_i at w (buy cost + lot penalty)
    double plo, phi_;
    const double s = -dw;                         // sell amount
    int nl = 0; const double *sl = nullptr, *wd = nullptr;
    if (LOTS) { nl = p.lot_count[row + i]; sl = p.lot_slope + (row + i) * L; wd = p.lot_width + (row + i) * L; }
    if (dw > dl) { plo = phi_ = cb; }
    else if (nl == 0) { if (s > dl) { plo = phi_ = 0.0; } else { plo = 0.0; phi_ = cb; } }
    else {
      // lots whose range [Q_l, Q_l + q_l] comes within delta of the sell amount s are "touched": the subdifferential
      // of the penalty is [-max touched slope, -min touched slope]; at s <= delta the buy side (c_buy) joins, at the
      // end of the last lot no further selling is possible (lower end -inf).
      double Q = 0.0, tax = 0.0, smin = INFINITY, smax = -INFINITY;
      for (int l = 0; l < nl; ++l) {
        const double ql = wd[l];
        tax += sl[l] * fmin(fmax(s - Q, 0.0), ql);
        if (s >= Q - dl && s <= Q + ql + dl) { smin = fmin(smin, sl[l]); smax = fmax(smax, sl[l]); }
        Q += ql;
      }
      plo = (s >= Q - dl) ? -INFINITY : -smax;
      phi_ = (s <= dl) ? cb : -smin;
      pen += tax;
      rbox = fmax(rbox, (w0 - Q) - w);            // cannot sell more than the lots held
    }
    fobj += 0.5 * x * gs - mu * w + pen;
    if (have) {
      const double g = gs - mu + nu + (G ? lam[p.group_id[i]] : 0.0);
      double Slo = (dw > dl ? lamt : -lamt) + plo;
      double Shi = (dw < -dl ? -lamt : lamt) + phi_;
      if (w <= lo + dl) Slo = -INFINITY;
      if (w >= hi - dl) Shi = INFINITY;
      rstat = fmax(rstat, fmax(fmax(Slo + g, -g - Shi), 0.0));
    }
  }
  __syncthreads();
  for (int g = tid; g < G; g += nt) gsum[g] = group_total(gbin, G, g);
  __syncthreads();
  double val[3] = {sw, turn, fobj};
  block_reduce<3, 0>(val, scratch);
  double vmx[2] = {rbox, rstat};
  block_reduce<2, 1>(vmx, scratch);
  const int any_bad = __syncthreads_or(bad ? 1 : 0);
  if (tid == 0) {
    double* r = p.resid + (int64_t)a * PRISM_NRES;
    const double nan = any_bad ? NAN : 0.0;
    r[PRISM_R_BUDGET] = fabs(val[0] - 1.0) + nan;
    r[PRISM_R_BOX] = fmax(vmx[0], 0.0) + nan;
    double rexp = 0.0, rcomp = 0.0;
    for (int g = 0; g < G; ++g) {
      const double bl = p.band_lo[(int64_t)a * G + g], bh = p.band_hi[(int64_t)a * G + g];
      rexp = fmax(rexp, fmax(bl - gsum[g], gsum[g] - bh));
      if (have) rcomp = fmax(rcomp, fmax(fabs(du[2 + g] * (gsum[g] - bh)), fabs(du[2 + G + g] * (bl - gsum[g]))));
    }
    r[PRISM_R_EXPOSURE] = fmax(rexp, 0.0);
    r[PRISM_R_TURNOVER] = isfinite(tau) ? fmax(val[1] - tau, 0.0) : 0.0;
    if (have && isfinite(tau)) rcomp = fmax(rcomp, fabs(theta * (val[1] - tau)));
    r[PRISM_R_STAT] = have ? vmx[1] : NAN;
    r[PRISM_R_COMP] = have ? rcomp : NAN;
    r[PRISM_R_OBJECTIVE] = val[2] + nan;
    r[PRISM_R_TURNOVER_VALUE] = val[1];
  }
}

// Status vocabulary (Table 14).  gates: self-imposed 1e-6 on all four feasibility residuals (reading R12).
__global__ void k_status(int A, const double* resid, const int32_t* conv, const int32_t* iters, int timed_out,
                         int late_iter, double gate, int32_t* status) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= A) return;
  const double* r = resid + (int64_t)a * PRISM_NRES;
  bool nanv = false;
  for (int c = 0; c < 4; ++c) nanv |= !(r[c] == r[c]);
  nanv |= !(r[PRISM_R_OBJECTIVE] == r[PRISM_R_OBJECTIVE]);
  const bool gates = r[PRISM_R_BUDGET] <= gate && r[PRISM_R_BOX] <= gate && r[PRISM_R_EXPOSURE] <= gate && r[PRISM_R_TURNOVER] <= gate;
  int s;
  if (conv[a] < 0 || nanv) s = PRISM_STATUS_FAILURE;
  else if (!gates) s = PRISM_STATUS_NO_FEASIBLE;
  else if (conv[a] == 1) s = (late_iter >= 0 && iters[a] > late_iter) ? PRISM_STATUS_LATE : PRISM_STATUS_CERTIFIED;
  else s = timed_out ? PRISM_STATUS_TIMEOUT : PRISM_STATUS_FEASIBLE;
  status[a] = s;
}
