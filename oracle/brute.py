"""TEST INFRASTRUCTURE ONLY - CPU oracle, never imported by the product path.

O-3 of SURVEY.md 8(c): brute-force active-set enumeration for tiny instances (N <= 6; N <= 4 with lots),
`BASELINE.json:north_star` ("brute-force active-set enumeration on tiny instances (N <= 6)").
Independent of the interior-point solver: no barrier, no lifting, dense Sigma.

Every coordinate is assigned a *piece* of its scalar cost: fixed at lo, at hi, at the kink w0, at an interior lot
breakpoint w0 - Q_l, or free on a linear piece (buy side, or inside sell lot l).  Every global inequality
(turnover cap, each band side) is either held at equality or dropped.  On such a face the objective of Eq. (1)
 is a strictly convex quadratic and the budget/active rows are linear equalities, so its minimiser
over the face is one linear solve.  The optimum w* of the full problem lies in the relative interior of exactly one
face and minimises the face's quadratic there, so w* is among the candidates; every candidate that satisfies all
constraints has f >= f(w*).  Hence

    w* = argmin { f(cand) : cand feasible }          (f evaluated by its definition, `problem.objective`)

No multiplier sign logic is needed, which is what makes this a pin and not a second solver.
"""
from __future__ import annotations

import itertools

import numpy as np

from .problem import Account, objective, sigma_dense


def _pieces(acc: Account, i: int):
    """List of (kind, value | None, slope, sgn) for coordinate i."""
    lo, hi, w0 = acc.lo[i], acc.hi[i], acc.w0[i]
    out = [("fix", lo, 0.0, 0.0)]
    if hi > lo:
        out.append(("fix", hi, 0.0, 0.0))
    else:
        return out
    if lo < w0 < hi:
        out.append(("fix", w0, 0.0, 0.0))
    if hi > w0:
        out.append(("free", None, acc.c_buy, +1.0))
    Li = int(acc.lot_count[i]) if acc.lot_slope is not None else 0
    if Li == 0:
        if lo < w0:
            out.append(("free", None, 0.0, -1.0))
    else:
        Q = 0.0
        for l in range(Li):
            out.append(("free", None, -acc.lot_slope[i, l], -1.0))
            Q += acc.lot_width[i, l]
            bp = w0 - Q
            if lo < bp < hi:
                out.append(("fix", bp, 0.0, 0.0))
    return out


def solve(acc: Account, feas_tol: float = 1e-10):
    N = acc.N
    Sig = sigma_dense(acc)
    wb = np.zeros(N) if acc.w_b is None else acc.w_b
    pieces = [_pieces(acc, i) for i in range(N)]
    has_tau = np.isfinite(acc.tau)
    G = acc.G
    E = np.zeros((G, N))
    if G > 0:
        E[acc.group_id, np.arange(N)] = 1.0
    floor = acc.lo.copy()
    if acc.lot_slope is not None:
        from .problem import sell_floor
        floor = sell_floor(acc)
    glob = [(False, True) if has_tau else (False,)] + [(0, 1, 2)] * G      # band: 0 inactive, 1 upper, 2 lower
    best = (np.inf, None)
    n_cand = 0
    for combo in itertools.product(*pieces):
        free = np.array([c[0] == "free" for c in combo])
        F = np.nonzero(free)[0]
        w_fix = np.array([0.0 if c[1] is None else c[1] for c in combo])
        slope = np.array([c[2] for c in combo]); sgn = np.array([c[3] for c in combo])
        nF = len(F)
        for gsel in itertools.product(*glob):
            tact = gsel[0]
            bact = [(g, gsel[1 + g]) for g in range(G) if gsel[1 + g] != 0]
            rows = [np.ones(nF)]
            rhs = [acc.budget - w_fix[~free].sum()]
            if tact:
                # sum_fixed dt |w - w0| + sum_free sgn dt (w - w0) = tau
                rows.append((sgn * acc.dt)[F])
                rhs.append(acc.tau - np.sum(acc.dt[~free] * np.abs(w_fix[~free] - acc.w0[~free])) + np.sum((sgn * acc.dt * acc.w0)[F]))
            for g, side in bact:
                rows.append(E[g, F])
                rhs.append((acc.band_hi[g] if side == 1 else acc.band_lo[g]) - E[g, ~free] @ w_fix[~free])
            nc = len(rows)
            if nc > nF + 0 and nF == 0:
                # nothing free: candidate is w_fix itself, equality rows must already hold
                w = w_fix
            else:
                if nc > nF:
                    continue
                C = np.array(rows).reshape(nc, nF)
                K = np.zeros((nF + nc, nF + nc))
                K[:nF, :nF] = acc.gamma * Sig[np.ix_(F, F)]
                K[:nF, nF:] = C.T; K[nF:, :nF] = C
                lin = (acc.mu + acc.gamma * (Sig @ wb))[F] - acc.gamma * (Sig[np.ix_(F, np.nonzero(~free)[0])] @ w_fix[~free]) \
                    - slope[F] - sgn[F] * acc.kappa * acc.dt[F]
                try:
                    sol = np.linalg.solve(K, np.concatenate([lin, rhs]))
                except np.linalg.LinAlgError:
                    continue
                w = w_fix.copy(); w[F] = sol[:nF]
            n_cand += 1
            # feasibility of the candidate for the FULL problem
            if abs(w.sum() - acc.budget) > feas_tol: continue
            if np.any(w < floor - feas_tol) or np.any(w > acc.hi + feas_tol): continue
            if has_tau and np.sum(acc.dt * np.abs(w - acc.w0)) > acc.tau + feas_tol: continue
            if G > 0:
                gs = E @ w
                if np.any(gs > acc.band_hi + feas_tol) or np.any(gs < acc.band_lo - feas_tol): continue
            fval = objective(acc, w, dense=True)
            if fval < best[0]:
                best = (fval, w.copy())
    return dict(w=best[1], f=best[0], n_candidates=n_cand)
