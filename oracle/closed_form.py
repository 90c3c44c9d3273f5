"""TEST INFRASTRUCTURE ONLY - CPU oracle, never imported by the product path.

Closed forms and textbook routines that pin the oracle (SURVEY.md 8(c) "Pins"):

* budget only (`BASELINE.json:north_star`): w = Sigma^-1 (mu/gamma + lambda 1), lambda from 1'w = 1
  (stationarity gamma Sigma w - mu - nu 1 = 0 of Eq. (1), with only the budget row).
* diagonal risk (B = 0), box + budget: the separable continuous quadratic knapsack,
  w_i = clip((mu_i - nu)/(gamma d_i), lo_i, hi_i) with nu by bisection on 1'w = 1.
* gamma Sigma = I, box + budget: Euclidean projection of mu onto the capped simplex (sort-based).
"""
from __future__ import annotations

import numpy as np

from .problem import Account, sigma_dense


def budget_only(acc: Account) -> np.ndarray:
    Sig = sigma_dense(acc)
    L = np.linalg.cholesky(Sig)

    def sinv(b):
        return np.linalg.solve(L.T, np.linalg.solve(L, b))
    rhs = acc.mu / acc.gamma
    if acc.w_b is not None:
        rhs = rhs + Sig @ acc.w_b
    a = sinv(rhs); o = sinv(np.ones(acc.N))
    lam = (acc.budget - a.sum()) / o.sum()
    return a + lam * o


def separable_knapsack(mu, gd, lo, hi, budget=1.0, iters=200):
    """min sum gd_i/2 w_i^2 - mu_i w_i  s.t. sum w = budget, lo <= w <= hi  (bisection on the multiplier)."""
    def w_of(nu):
        return np.clip((mu - nu) / gd, lo, hi)
    a = float(np.min(mu - gd * hi)) - 1.0
    b = float(np.max(mu - gd * lo)) + 1.0
    for _ in range(iters):
        m = 0.5 * (a + b)
        if w_of(m).sum() > budget:
            a = m
        else:
            b = m
    return w_of(0.5 * (a + b))


def capped_simplex_projection(v, cap, budget=1.0):
    """argmin ||w - v||^2 s.t. sum w = budget, 0 <= w <= cap: exact search over the sorted breakpoints."""
    bps = np.sort(np.concatenate([v, v - cap]))
    # s(t) = sum clip(v - t, 0, cap) is piecewise linear, non-increasing in t
    def s(t):
        return np.clip(v - t, 0.0, cap).sum()
    lo_i, hi_i = 0, len(bps) - 1
    if s(bps[0]) < budget:
        raise ValueError("infeasible")
    while hi_i - lo_i > 1:
        mid = (lo_i + hi_i) // 2
        if s(bps[mid]) >= budget:
            lo_i = mid
        else:
            hi_i = mid
    t0, t1 = bps[lo_i], bps[hi_i]
    s0, s1 = s(t0), s(t1)
    t = t0 if s0 == s1 else t0 + (s0 - budget) * (t1 - t0) / (s0 - s1)
    return np.clip(v - t, 0.0, cap)
