"""Hand-computed fixtures under tests/golden/ (each file carries its derivation and citation)."""
import os

import numpy as np

from oracle import ipm, problem

HERE = os.path.dirname(os.path.abspath(__file__))


def _rows():
    out = {}
    with open(os.path.join(HERE, "golden", "two_asset_closed_form.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                p = line.split()
                out[p[0]] = [float(x) for x in p[1:]]
    return out


def _account(gamma, d, mu, w0, **kw):
    N = len(d)
    base = dict(N=N, B=np.zeros((N, 1)), f=np.ones(1), d=np.array(d), mu=np.array(mu), gamma=gamma, w0=np.array(w0), w_b=None,
                lo=np.full(N, -10.0), hi=np.full(N, 10.0), dt=np.ones(N), tau=np.inf, kappa=0.0, c_buy=0.0, group_id=None, G=0,
                band_lo=None, band_hi=None, lot_slope=None, lot_width=None, lot_count=None)
    base.update(kw)
    return problem.Account(**base)


def test_two_asset_budget_only():
    gamma, d1, d2, mu1, mu2, w1, w2, fval, nu = _rows()["A"]
    acc = _account(gamma, [d1, d2], [mu1, mu2], [0.5, 0.5])
    r = ipm.solve(acc, mode="dense")
    assert r["status"] == "optimal"
    assert np.allclose(r["w"], [w1, w2], atol=1e-10)
    assert abs(problem.objective(acc, np.array([w1, w2])) - fval) < 1e-15
    assert abs(r["mult"]["nu"] - nu) < 1e-9


def test_lot_penalty_definition():
    s1, s2, q1, q2, sell, psi = _rows()["B"]
    acc = _account(1.0, [0.01], [0.0], [0.3], lot_slope=np.array([[s1, s2, 0, 0]]), lot_width=np.array([[q1, q2, 0, 0]]),
                   lot_count=np.array([2]))
    assert abs(problem.tax_sell_penalty(acc, np.array([sell]))[0] - psi) < 1e-16
