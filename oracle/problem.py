"""TEST INFRASTRUCTURE ONLY - CPU oracle, never imported by the product path.

Per-account view of Eq. (1) in the concretisation of SURVEY.md 8.0:

    minimise   (gamma/2) (w-w_b)' Sigma (w-w_b) - mu'w
               + kappa * sum_i dt_i |w_i - w0_i|
               + sum_i [ c_buy (w_i-w0_i)_+ + psi_i((w0_i-w_i)_+) ]
    subject to 1'w = 1,  lo <= w <= hi,  band_lo <= E w <= band_hi,  sum_i dt_i |w_i-w0_i| <= tau
    Sigma = B diag(f) B' + diag(d)
    psi_i(s) = sum_l slope_il * min(max(s - Q_{i,l-1}, 0), width_il)      (convex: slopes ascend)

`objective` is that definition written out in fp64 (dense Sigma when asked, factor form otherwise).
Everything here depends only on numpy and on the data container of `instances.gen`.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np


@dataclass
class Account:
    """Problem data of one account, plain arrays (fp64)."""
    N: int
    B: np.ndarray            # (N, k)
    f: np.ndarray            # (k,)
    d: np.ndarray            # (N,)
    mu: np.ndarray           # (N,)
    gamma: float
    w0: np.ndarray           # (N,)
    w_b: Optional[np.ndarray]
    lo: np.ndarray           # (N,)
    hi: np.ndarray           # (N,)
    dt: np.ndarray           # (N,)
    tau: float               # inf => no cap
    kappa: float
    c_buy: float
    group_id: Optional[np.ndarray]   # (N,) ints in 0..G-1
    G: int
    band_lo: Optional[np.ndarray]    # (G,)
    band_hi: Optional[np.ndarray]
    lot_slope: Optional[np.ndarray]  # (N, L)
    lot_width: Optional[np.ndarray]  # (N, L)
    lot_count: Optional[np.ndarray]  # (N,)
    budget: float = 1.0


def account_from_instance(inst, a: int) -> Account:
    lo, hi = inst.bounds(a)
    return Account(
        N=inst.N, B=inst.B, f=inst.f, d=inst.d, mu=inst.mu[a], gamma=float(inst.gamma[a]),
        w0=inst.w0[a], w_b=None if inst.w_b is None else inst.w_b[a], lo=lo, hi=hi,
        dt=np.ones(inst.N) if inst.d_t is None else inst.d_t, tau=float(inst.tau[a]),
        kappa=float(inst.kappa[a]), c_buy=float(inst.c_buy[a]),
        group_id=None if inst.group_id is None else inst.group_id.astype(np.int64), G=inst.G,
        band_lo=None if inst.band_lo is None else inst.band_lo[a],
        band_hi=None if inst.band_hi is None else inst.band_hi[a],
        lot_slope=None if inst.lot_slope is None else inst.lot_slope[a],
        lot_width=None if inst.lot_width is None else inst.lot_width[a],
        lot_count=None if inst.lot_count is None else inst.lot_count[a].astype(np.int64),
    )


def sigma_dense(acc: Account) -> np.ndarray:
    """Sigma = B F B' + D materialised (PAPER.md:128 'factor-structured risk')."""
    return (acc.B * acc.f) @ acc.B.T + np.diag(acc.d)


def sigma_apply(acc: Account, x: np.ndarray) -> np.ndarray:
    return acc.B @ (acc.f * (acc.B.T @ x)) + acc.d * x


def tax_sell_penalty(acc: Account, sell: np.ndarray) -> np.ndarray:
    """psi_i(sell_i) per asset, by the definition above (one term per lot, in lot order)."""
    out = np.zeros(acc.N)
    if acc.lot_slope is None:
        return out
    L = acc.lot_slope.shape[1]
    Qprev = np.zeros(acc.N)
    for l in range(L):
        live = acc.lot_count > l
        fill = np.minimum(np.maximum(sell - Qprev, 0.0), acc.lot_width[:, l])
        out += np.where(live, acc.lot_slope[:, l] * fill, 0.0)
        Qprev = Qprev + np.where(live, acc.lot_width[:, l], 0.0)
    return out


def objective(acc: Account, w: np.ndarray, dense: bool = False) -> float:
    """f(w) of SURVEY.md 8.0 (the public objective of Eq. (1))."""
    x = w if acc.w_b is None else w - acc.w_b
    if dense:
        risk = 0.5 * acc.gamma * float(x @ (sigma_dense(acc) @ x))
    else:
        s = acc.B.T @ x
        risk = 0.5 * acc.gamma * (float(np.sum(acc.f * s * s)) + float(np.sum(acc.d * x * x)))
    dw = w - acc.w0
    val = risk - float(acc.mu @ w)
    val += acc.kappa * float(np.sum(acc.dt * np.abs(dw)))
    val += acc.c_buy * float(np.sum(np.maximum(dw, 0.0)))
    val += float(np.sum(tax_sell_penalty(acc, np.maximum(-dw, 0.0))))
    return val


def turnover(acc: Account, w: np.ndarray) -> float:
    return float(np.sum(acc.dt * np.abs(w - acc.w0)))


def group_sums(acc: Account, w: np.ndarray) -> np.ndarray:
    if acc.G == 0:
        return np.zeros(0)
    return np.bincount(acc.group_id, weights=w, minlength=acc.G)


def sell_floor(acc: Account) -> np.ndarray:
    """Lowest weight reachable by selling: lo, and with lots also w0 - (sum of lot widths)."""
    if acc.lot_slope is None:
        return acc.lo.copy()
    L = acc.lot_slope.shape[1]
    live = np.arange(L)[None, :] < acc.lot_count[:, None]
    Q = np.sum(np.where(live, acc.lot_width, 0.0), axis=1)
    has = acc.lot_count > 0
    return np.where(has, np.maximum(acc.lo, acc.w0 - Q), acc.lo)
