"""TEST INFRASTRUCTURE ONLY - CPU oracle, never imported by the product path.

K-check of SURVEY.md 8(c): the paper's external diagnostics written out literally, in a file of its own
(it shares no code with `ipm.py`):

  feasibility (Section 4.4)
      r_budget   = |1'w - 1|
      r_box      = max(||(lo - w)_+||_inf, ||(w - hi)_+||_inf)
      r_exposure = max(||(b_min - A w)_+||_inf, ||(A w - b_max)_+||_inf)       (A = group indicator rows)
      r_turnover = (||D (w - w0)||_1 - tau)_+
  KKT-style, constraints g_i(w) <= 0 with multipliers lambda_i >= 0, budget multiplier nu:
      r_stat = || grad f + sum_i lambda_i grad g_i + nu 1 ||_inf
      r_comp = max_i |lambda_i g_i(w)|
  For the nonsmooth terms of the public objective (L1 transition, buy cost, piecewise-linear lot penalty) and the
  box, "grad" is read as the subgradient-distance form (reading R19): per asset the set
      S_i = (kappa+theta) dt_i d|w_i - w0_i| + d phi_i(w_i) + N_[lo_i,hi_i](w_i)
  is a closed interval and r_stat = max_i dist(-g_i, S_i),  g_i = [gamma Sigma (w - w_b) - mu + nu 1 + E'(lam_hi - lam_lo)]_i.
  Activity is decided with delta = 1e-9.

`certify_free` is the multiplier-free variant: it minimises r_stat over (nu, theta >= 0, lam >= 0) as a small LP
(complementarity imposed by fixing multipliers of inactive constraints to zero), so a weight vector can be
certified without any solver's duals.
"""
from __future__ import annotations

import numpy as np

from .problem import Account, sigma_apply

DELTA = 1e-9


def feasibility(acc: Account, w: np.ndarray) -> dict:
    r_budget = abs(float(np.sum(w)) - acc.budget)
    r_box = max(float(np.max(np.maximum(acc.lo - w, 0.0))), float(np.max(np.maximum(w - acc.hi, 0.0))))
    if acc.lot_slope is not None:           # sells cannot exceed the lots held (w >= w0 - sum of widths)
        L = acc.lot_slope.shape[1]
        live = np.arange(L)[None, :] < acc.lot_count[:, None]
        Q = np.sum(np.where(live, acc.lot_width, 0.0), axis=1)
        has = acc.lot_count > 0
        r_box = max(r_box, float(np.max(np.where(has, np.maximum(acc.w0 - Q - w, 0.0), 0.0))))
    r_exp = 0.0
    if acc.G > 0:
        gs = np.bincount(acc.group_id, weights=w, minlength=acc.G)
        r_exp = max(float(np.max(np.maximum(acc.band_lo - gs, 0.0))), float(np.max(np.maximum(gs - acc.band_hi, 0.0))))
    r_turn = 0.0
    if np.isfinite(acc.tau):
        r_turn = max(float(np.sum(acc.dt * np.abs(w - acc.w0))) - acc.tau, 0.0)
    return dict(r_budget=r_budget, r_box=r_box, r_exposure=r_exp, r_turnover=r_turn)


def _phi_interval(acc: Account, w: np.ndarray, delta: float):
    """Subdifferential [lo, hi] of phi_i(w_i) = c_buy (w_i-w0_i)_+ + psi_i((w0_i-w_i)_+) per asset."""
    N = acc.N
    dw = w - acc.w0
    lo = np.empty(N); hi = np.empty(N)
    buy = dw > delta
    lo[buy] = acc.c_buy; hi[buy] = acc.c_buy
    if acc.lot_slope is None:
        sell = dw < -delta
        lo[sell] = 0.0; hi[sell] = 0.0
        kink = ~buy & ~sell
        lo[kink] = 0.0; hi[kink] = acc.c_buy
        return lo, hi
    L = acc.lot_slope.shape[1]
    for i in range(N):
        if buy[i]:
            continue
        s = -dw[i]                       # sell amount >= -delta
        Li = int(acc.lot_count[i])
        if Li == 0:
            if s > delta:
                lo[i] = hi[i] = 0.0
            else:
                lo[i], hi[i] = 0.0, acc.c_buy
            continue
        # derivative of phi wrt w on the sell side is -slope of the lot being consumed.  Activity with threshold
        # delta (reading R19): every lot whose range [Q_l, Q_l + q_l] comes within delta of s is "touched" (lots can
        # be narrower than delta), and the subdifferential is [-max touched slope, -min touched slope]; at s <= delta
        # the buy side joins (upper end c_buy); at the end of the last lot no further selling is possible (-inf).
        Q = 0.0
        touched = []
        for l in range(Li):
            q = acc.lot_width[i, l]
            if Q - delta <= s <= Q + q + delta:
                touched.append(acc.lot_slope[i, l])
            Q += q
        lo[i] = -np.inf if s >= Q - delta else -max(touched)
        hi[i] = acc.c_buy if s <= delta else -min(touched)
    return lo, hi


def _intervals(acc: Account, w: np.ndarray, theta: float, delta: float):
    lam = acc.kappa + theta
    dw = w - acc.w0
    a_lo = np.where(dw > delta, lam * acc.dt, -lam * acc.dt)
    a_hi = np.where(dw < -delta, -lam * acc.dt, lam * acc.dt)
    p_lo, p_hi = _phi_interval(acc, w, delta)
    S_lo = a_lo + p_lo; S_hi = a_hi + p_hi
    at_lo = w <= acc.lo + delta; at_hi = w >= acc.hi - delta
    S_lo = np.where(at_lo, -np.inf, S_lo)
    S_hi = np.where(at_hi, np.inf, S_hi)
    return S_lo, S_hi


def kkt(acc: Account, w: np.ndarray, mult: dict, delta: float = DELTA) -> dict:
    """r_stat and r_comp for given multipliers nu, theta, lam_hi, lam_lo."""
    x = w if acc.w_b is None else w - acc.w_b
    g = acc.gamma * sigma_apply(acc, x) - acc.mu + mult["nu"]
    gs = None
    if acc.G > 0:
        g = g + (np.asarray(mult["lam_hi"]) - np.asarray(mult["lam_lo"]))[acc.group_id]
        gs = np.bincount(acc.group_id, weights=w, minlength=acc.G)
    theta = float(mult.get("theta", 0.0))
    S_lo, S_hi = _intervals(acc, w, theta, delta)
    dist = np.maximum(np.maximum(S_lo - (-g), (-g) - S_hi), 0.0)
    r_stat = float(np.max(dist))
    r_comp = 0.0
    if np.isfinite(acc.tau):
        r_comp = max(r_comp, abs(theta * (float(np.sum(acc.dt * np.abs(w - acc.w0))) - acc.tau)))
    if acc.G > 0:
        r_comp = max(r_comp, float(np.max(np.abs(np.asarray(mult["lam_hi"]) * (gs - acc.band_hi)))),
                     float(np.max(np.abs(np.asarray(mult["lam_lo"]) * (acc.band_lo - gs)))))
    neg = min(theta, 0.0)
    if acc.G > 0:
        neg = min(neg, float(np.min(mult["lam_hi"])), float(np.min(mult["lam_lo"])))
    return dict(r_stat=r_stat, r_comp=r_comp, min_multiplier=neg, worst=int(np.argmax(dist)))


def certify_free(acc: Account, w: np.ndarray, delta: float = DELTA, act_tol: float = 1e-7) -> dict:
    """Multiplier-free certificate: min_{nu, theta>=0, lam>=0} r_stat as an LP (scipy HiGHS)."""
    from scipy.optimize import linprog
    x = w if acc.w_b is None else w - acc.w_b
    g0 = acc.gamma * sigma_apply(acc, x) - acc.mu
    G = acc.G
    # variables: [t, nu, theta, lam_hi (G), lam_lo (G)]
    nvar = 3 + 2 * G
    S_lo0, S_hi0 = _intervals(acc, w, 0.0, delta)            # theta enters linearly on top of these
    dw = w - acc.w0
    c_lo = np.where(dw > delta, acc.dt, -acc.dt)             # d S_lo / d theta
    c_hi = np.where(dw < -delta, -acc.dt, acc.dt)
    rows = []; rhs = []
    E = np.zeros((acc.N, G))
    if G > 0:
        E[np.arange(acc.N), acc.group_id] = 1.0
    # S_lo0 + theta c_lo - t <= -(g0 + nu + E(lam_hi - lam_lo))   (only where S_lo finite)
    m = np.isfinite(S_lo0)
    A1 = np.zeros((int(m.sum()), nvar)); A1[:, 0] = -1.0; A1[:, 1] = 1.0; A1[:, 2] = c_lo[m]
    A1[:, 3:3 + G] = E[m]; A1[:, 3 + G:] = -E[m]
    rows.append(A1); rhs.append(-g0[m] - S_lo0[m])
    m = np.isfinite(S_hi0)
    A2 = np.zeros((int(m.sum()), nvar)); A2[:, 0] = -1.0; A2[:, 1] = -1.0; A2[:, 2] = -c_hi[m]
    A2[:, 3:3 + G] = -E[m]; A2[:, 3 + G:] = E[m]
    rows.append(A2); rhs.append(g0[m] + S_hi0[m])
    bounds = [(0, None), (None, None)]
    turn_active = np.isfinite(acc.tau) and abs(float(np.sum(acc.dt * np.abs(dw))) - acc.tau) <= act_tol
    bounds.append((0, None) if turn_active else (0, 0))
    if G > 0:
        gs = np.bincount(acc.group_id, weights=w, minlength=G)
        for g in range(G):
            bounds.append((0, None) if abs(gs[g] - acc.band_hi[g]) <= act_tol else (0, 0))
        for g in range(G):
            bounds.append((0, None) if abs(gs[g] - acc.band_lo[g]) <= act_tol else (0, 0))
    cost = np.zeros(nvar); cost[0] = 1.0
    res = linprog(cost, A_ub=np.vstack(rows), b_ub=np.concatenate(rhs), bounds=bounds, method="highs")
    if res.status != 0:
        return dict(r_stat=np.inf, ok=False)
    z = res.x
    return dict(r_stat=float(z[0]), ok=True, nu=float(z[1]), theta=float(z[2]), lam_hi=z[3:3 + G], lam_lo=z[3 + G:])


def distance_bound(acc: Account, gap: float) -> float:
    """||w - w*||_2 <= sqrt(2 gap / m), m = gamma min_i d_i the strong-convexity modulus."""
    return float(np.sqrt(2.0 * max(gap, 0.0) / (acc.gamma * float(np.min(acc.d)))))
