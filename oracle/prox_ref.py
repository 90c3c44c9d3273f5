"""TEST INFRASTRUCTURE ONLY - CPU oracle, never imported by the product path.

The proximal / projection step of the splitting by its DEFINITION, for the prox-only parity test
("kernel vs a 1-D restatement on random v"):

    prox(v; rho) = argmin_z  sum_i rho_i / 2 (z_i - v_i)^2 + kappa dt_i |z_i - w0_i| + c_buy (z_i - w0_i)_+ + psi_i((w0_i - z_i)_+)
                   s.t.  1'z = 1,  lo <= z <= hi,  band_lo <= E z <= band_hi,  sum_i dt_i |z_i - w0_i| <= tau
    (every nonsmooth / polyhedral term of Eq. (1), in the metric diag(rho)).

Two independent routes:

* `prox_qp`      - the prox problem IS an instance of Eq. (1) with a diagonal risk matrix: gamma = 1, B = 0, D = diag(rho),
                   mu = rho o v, since sum rho/2 (z - v)^2 = 1/2 z'diag(rho)z - (rho o v)'z + const.  It is handed to the
                   interior-point oracle (ipm.py) unchanged; every constraint family (bands, lots, caps) is covered.
* `prox_nested`  - no bands, no lots: the definition through its Lagrangian, written with one-dimensional searches only
                   (no formula of the kernel is restated).  For multipliers (nu, theta) of budget and turnover cap each
                   asset minimises its own scalar convex function  rho/2 (z-v)^2 + (kappa+theta) dt |z-w0| + c_buy (z-w0)_+ - nu z
                   over [lo, hi] by golden-section search; nu is found by bisection on the budget (sum z is
                   non-decreasing in nu), theta >= 0 by bisection on the turnover (non-increasing in theta), 0 if the cap
                   is slack.  Accuracy ~1e-8 (golden section on a function that is flat at its minimum); pins prox_qp.
Pins: tests/test_oracle_pins.py::test_prox_reference_* (prox_qp == prox_nested on small cases; capped-simplex special
case against the textbook sort-based projection; kkt_check certificate of the prox problem).
"""
from __future__ import annotations

import dataclasses

import numpy as np

from . import ipm
from .problem import Account


def prox_problem(acc: Account, v: np.ndarray, rho: np.ndarray) -> Account:
    """The prox at v as an Eq. (1) instance: gamma = 1, Sigma = diag(rho), mu = rho o v, no benchmark shift."""
    return dataclasses.replace(acc, B=np.zeros((acc.N, 1)), f=np.ones(1), d=np.asarray(rho, dtype=np.float64).copy(),
                               mu=np.asarray(rho * v, dtype=np.float64), gamma=1.0, w_b=None)


def prox_qp(acc: Account, v: np.ndarray, rho: np.ndarray, witness=None) -> dict:
    """prox(v; rho) through the interior-point oracle on `prox_problem`; returns ipm.solve's dict (w = the prox)."""
    return ipm.solve(prox_problem(acc, v, rho), witness=witness)


def _golden(fun, lo, hi, steps=90):
    """Vectorised golden-section minimisation of the scalar convex functions fun(z)[i] over [lo[i], hi[i]]."""
    g = 0.5 * (np.sqrt(5.0) - 1.0)
    a, b = lo.astype(np.float64).copy(), hi.astype(np.float64).copy()
    c, d = b - g * (b - a), a + g * (b - a)
    fc, fd = fun(c), fun(d)
    for _ in range(steps):
        left = fc < fd
        b = np.where(left, d, b); a = np.where(left, a, c)
        c_new = b - g * (b - a); d_new = a + g * (b - a)
        c, d = c_new, d_new
        fc, fd = fun(c), fun(d)
    return 0.5 * (a + b)


def prox_nested(acc: Account, v: np.ndarray, rho: np.ndarray, outer=70) -> np.ndarray:
    assert acc.G == 0 and acc.lot_slope is None, "prox_nested: no bands, no lots"
    w0, dt = acc.w0, acc.dt

    def z_of(nu, theta):
        def fun(z):
            t = z - w0
            return 0.5 * rho * (z - v) ** 2 + (acc.kappa + theta) * dt * np.abs(t) + acc.c_buy * np.maximum(t, 0.0) - nu * z
        return _golden(fun, acc.lo, acc.hi)

    span = float(np.max(rho * (np.abs(v) + np.abs(acc.hi) + np.abs(acc.lo) + 1.0))) + acc.kappa + acc.c_buy + 1.0

    def solve_nu(theta):
        lo_n, hi_n = -span - theta * float(np.max(dt)), span + theta * float(np.max(dt))
        for _ in range(outer):
            mid = 0.5 * (lo_n + hi_n)
            if float(np.sum(z_of(mid, theta))) < acc.budget:
                lo_n = mid
            else:
                hi_n = mid
        return z_of(0.5 * (lo_n + hi_n), theta)

    z = solve_nu(0.0)
    if not np.isfinite(acc.tau) or float(np.sum(dt * np.abs(z - w0))) <= acc.tau:
        return z
    lo_t, hi_t = 0.0, 2.0 * span
    for _ in range(outer):
        mid = 0.5 * (lo_t + hi_t)
        if float(np.sum(dt * np.abs(solve_nu(mid) - w0))) > acc.tau:
            lo_t = mid
        else:
            hi_t = mid
    return solve_nu(hi_t)
