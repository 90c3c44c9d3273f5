"""Pins of the CPU oracle (SURVEY.md 8(c) "Pins"): the oracle is checked against things other than itself -
the budget-only closed form (BASELINE.json:north_star), brute-force face enumeration on tiny instances,
textbook special cases (separable knapsack, capped-simplex projection), turnover cap/penalty duality,
invariances, and independent KKT certificates.  No GPU needed."""
import numpy as np
import pytest

from instances import gen
from oracle import brute, closed_form, ipm, kkt_check, problem


def _acc(inst, a=0):
    return problem.account_from_instance(inst, a)


def _solve(inst, a=0, mode="dense"):
    acc = _acc(inst, a)
    r = ipm.solve(acc, mode=mode, witness=inst.witness[a])
    assert r["status"] == "optimal", r["status"]
    return acc, r


def _certify(acc, r, tol=1e-8, delta=1e-7):
    feas = kkt_check.feasibility(acc, r["w"])
    assert max(feas.values()) <= 1e-9, feas
    k = kkt_check.kkt(acc, r["w"], r["mult"], delta=delta)
    assert k["r_stat"] <= tol and k["r_comp"] <= tol and k["min_multiplier"] >= -1e-12, k


# ---------------------------------------------------------------------------------- closed form
@pytest.mark.parametrize("seed", range(4))
def test_budget_only_closed_form(seed):
    """w = Sigma^-1 (mu/gamma + lambda 1), lambda from 1'w = 1 (north_star); box and cap made slack."""
    inst = gen.make_instance("bo", seed, 40, 5, 1, hi_fixed=50.0)
    inst.lo[:] = -50.0
    acc, r = _solve(inst)
    w_cf = closed_form.budget_only(acc)
    assert abs(w_cf.sum() - 1.0) < 1e-12
    assert np.max(np.abs(r["w"] - w_cf)) < 1e-9
    assert abs(problem.objective(acc, r["w"]) - problem.objective(acc, w_cf, dense=True)) < 1e-12


def test_budget_only_with_benchmark_shift():
    inst = gen.make_instance("bo_wb", 3, 30, 4, 1, hi_fixed=50.0, benchmark_in_risk=True)
    inst.lo[:] = -50.0
    acc, r = _solve(inst)
    assert np.max(np.abs(r["w"] - closed_form.budget_only(acc))) < 1e-9


# ---------------------------------------------------------------------------------- brute force
FAMILIES = {
    "box_cap": dict(N=5, kw=dict(hi_range=(0.3, 0.6), tau_range=(0.05, 0.6))),
    "exclusion": dict(N=5, kw=dict(hi_range=(0.35, 0.6), tau_range=(0.05, 0.6), excl_frac=0.2)),
    "l1_penalty": dict(N=5, kw=dict(hi_range=(0.3, 0.6), tau_range=(0.3, 0.9), kappa_fixed=0.01)),
    "penalty_only": dict(N=6, kw=dict(hi_range=(0.3, 0.6), kappa_fixed=0.005)),
    "buy_cost": dict(N=5, kw=dict(hi_range=(0.3, 0.6), tau_range=(0.1, 0.6), c_buy=0.003)),
    "lots": dict(N=4, kw=dict(hi_range=(0.4, 0.8), tau_range=(0.1, 0.8), lots=True, c_buy=5e-4)),
    "lots_caps": dict(N=4, kw=dict(hi_range=(0.5, 0.8), tau_range=(0.2, 0.8), lots=True, c_buy=5e-4, cap_frac=0.25,
                                   cap_range=(0.05, 0.3))),
    "bands": dict(N=5, kw=dict(hi_range=(0.3, 0.6), tau_range=(0.1, 0.8), G=2, band_half=0.02)),
}


@pytest.mark.parametrize("family", sorted(FAMILIES))
@pytest.mark.parametrize("seed", range(5))
def test_brute_force_enumeration(family, seed):
    """IPM = brute-force face enumeration (O-3) on tiny instances, every constraint family."""
    spec = FAMILIES[family]
    inst = gen.make_instance(family, 100 + seed, spec["N"], 2, 1, **spec["kw"])
    acc, r = _solve(inst)
    b = brute.solve(acc)
    assert b["w"] is not None
    assert np.max(np.abs(r["w"] - b["w"])) < 5e-8, (r["w"], b["w"])
    assert abs(problem.objective(acc, r["w"], dense=True) - b["f"]) < 1e-10
    _certify(acc, r)
    c = kkt_check.certify_free(acc, r["w"], delta=1e-7)
    assert c["ok"] and c["r_stat"] < 1e-7


# ---------------------------------------------------------------------------------- textbook special cases
@pytest.mark.parametrize("seed", range(3))
def test_diagonal_risk_is_separable_knapsack(seed):
    inst = gen.make_instance("diag", seed, 60, 3, 1, hi_fixed=0.08)
    inst.B[:] = 0.0
    acc, r = _solve(inst)
    w_ref = closed_form.separable_knapsack(acc.mu, acc.gamma * acc.d, acc.lo, acc.hi)
    assert np.max(np.abs(r["w"] - w_ref)) < 1e-8


@pytest.mark.parametrize("seed", range(3))
def test_identity_risk_is_capped_simplex_projection(seed):
    inst = gen.make_instance("proj", seed, 50, 3, 1, hi_fixed=0.07, gamma_fixed=1.0)
    inst.B[:] = 0.0
    inst.d[:] = 1.0
    rng = np.random.default_rng(seed)
    inst.mu[0] = rng.normal(0.0, 0.05, inst.N)
    acc, r = _solve(inst)
    w_ref = closed_form.capped_simplex_projection(acc.mu, 0.07)
    assert abs(w_ref.sum() - 1.0) < 1e-12
    assert np.max(np.abs(r["w"] - w_ref)) < 1e-8


# ---------------------------------------------------------------------------------- turnover cap
def test_turnover_cap_limits_and_monotone_value():
    inst = gen.make_instance("tau", 5, 40, 4, 1, hi_fixed=0.2, tau_fixed=0.3)
    acc = _acc(inst)
    vals = []
    for tau in [1e-7, 0.05, 0.1, 0.2, 0.4, 0.8, 5.0]:
        acc.tau = tau
        r = ipm.solve(acc, mode="dense", witness=acc.w0)
        assert r["status"] == "optimal"
        vals.append(problem.objective(acc, r["w"]))
        if tau == 1e-7:
            assert np.max(np.abs(r["w"] - acc.w0)) <= 1e-7          # tau -> 0 => w* = w0
        if tau == 5.0:
            w_big = r["w"]
    acc.tau = np.inf
    r = ipm.solve(acc, mode="dense", witness=acc.w0)
    assert np.max(np.abs(r["w"] - w_big)) < 1e-8                    # slack cap == no cap
    v = np.array(vals)
    assert np.all(np.diff(v) <= 1e-12)                                 # f*(tau) non-increasing
    taus = np.array([0.05, 0.1, 0.2, 0.4])
    # convexity of f*(tau) on the equally spaced-in-log sample: chord slopes increase
    sl = np.diff(v[1:5]) / np.diff(taus)
    assert np.all(np.diff(sl) >= -1e-10)


@pytest.mark.parametrize("seed", range(3))
def test_cap_penalty_duality(seed):
    """Solve with the cap -> theta*; re-solve with kappa = theta*, cap removed -> same w* (Lagrangian duality)."""
    inst = gen.make_instance("dual", seed, 50, 4, 1, hi_fixed=0.15, tau_fixed=0.25)
    acc, r = _solve(inst)
    theta = r["mult"]["theta"]
    assert theta > 1e-6
    acc2 = _acc(inst)
    acc2.tau = np.inf
    acc2.kappa = theta
    r2 = ipm.solve(acc2, mode="dense", witness=inst.witness[0])
    assert r2["status"] == "optimal"
    assert np.max(np.abs(r["w"] - r2["w"])) < 2e-7


# ---------------------------------------------------------------------------------- invariances
def test_scaling_and_permutation_invariance():
    inst = gen.make_instance("inv", 11, 40, 4, 1, hi_fixed=0.12, tau_fixed=0.3, kappa_fixed=0.002, lots=True, c_buy=5e-4)
    acc, r = _solve(inst)
    c = 3.7
    acc2 = _acc(inst)
    acc2.gamma *= c; acc2.mu = acc2.mu * c; acc2.kappa *= c; acc2.c_buy *= c; acc2.lot_slope = acc2.lot_slope * c
    r2 = ipm.solve(acc2, mode="dense", witness=inst.witness[0])
    assert np.max(np.abs(r["w"] - r2["w"])) < 1e-8
    assert abs(r2["mult"]["nu"] - c * r["mult"]["nu"]) < 1e-7
    perm = np.random.default_rng(0).permutation(inst.N)
    acc3 = _acc(inst)
    for name in ["mu", "w0", "lo", "hi", "dt", "d", "lot_count"]:
        setattr(acc3, name, getattr(acc3, name)[perm])
    acc3.B = acc3.B[perm]; acc3.lot_slope = acc3.lot_slope[perm]; acc3.lot_width = acc3.lot_width[perm]
    r3 = ipm.solve(acc3, mode="dense", witness=inst.witness[0][perm])
    assert np.max(np.abs(r["w"][perm] - r3["w"])) < 1e-8


# ---------------------------------------------------------------------------------- structured == dense
@pytest.mark.parametrize("name,builder", [
    ("cfg0", lambda: gen.config0()),
    ("cfg1", lambda: gen.config1(N=240, k=6, A=2)),
    ("cfg2", lambda: gen.config2(N=300, k=8, A=2, G=5, band_half=0.005)),
    ("cfg3", lambda: gen.config3(N=200, k=8, A=2)),
    ("cfg4", lambda: gen.config4(N=600, k=10, A=1, hi=0.004)),
    ("sec9", lambda: gen.section9(N=150, k=6, A=1)),
])
def test_structured_mode_equals_dense_mode(name, builder):
    inst = builder()
    for a in range(inst.A):
        acc, rd = _solve(inst, a, "dense")
        _, rs = _solve(inst, a, "structured")
        assert np.max(np.abs(rd["w"] - rs["w"])) < 2e-8
        _certify(acc, rs)
        gap = abs(problem.objective(acc, rs["w"]) - problem.objective(acc, rd["w"]))
        assert kkt_check.distance_bound(acc, gap) < 1e-3


# ---------------------------------------------------------------------------------- the checker itself
def test_checker_rejects_wrong_answers():
    inst = gen.config0()
    acc, r = _solve(inst)
    _certify(acc, r)
    w = r["w"].copy()
    i, j = np.argsort(-w)[:2]
    w[i] += 1e-4; w[j] -= 1e-4                                        # still budget-feasible, no longer optimal
    k = kkt_check.kkt(acc, w, r["mult"], delta=1e-7)
    assert k["r_stat"] > 1e-7 or kkt_check.feasibility(acc, w)["r_box"] > 0
    bad = dict(r["mult"]); bad["nu"] = r["mult"]["nu"] + 1e-3
    assert kkt_check.kkt(acc, r["w"], bad, delta=1e-7)["r_stat"] > 5e-4
    bad = dict(r["mult"]); bad["theta"] = r["mult"]["theta"] * 0.5
    assert kkt_check.kkt(acc, r["w"], bad, delta=1e-7)["r_stat"] > 1e-4
    w2 = r["w"] + 1e-3 / acc.N
    assert abs(kkt_check.feasibility(acc, w2)["r_budget"] - 1e-3) < 1e-12


def test_objective_factor_form_equals_dense_form():
    inst = gen.make_instance("obj", 2, 30, 4, 1, hi_fixed=0.2, tau_fixed=0.4, kappa_fixed=0.003, lots=True, c_buy=5e-4,
                             benchmark_in_risk=True)
    acc = _acc(inst)
    w = inst.witness[0]
    assert abs(problem.objective(acc, w) - problem.objective(acc, w, dense=True)) < 1e-14


# ---------------------------------------------------------------------------------- prox reference (oracle/prox_ref.py)
@pytest.mark.parametrize("seed,tau,kappa", [(0, 0.25, 0.0), (1, 0.05, 0.0), (2, np.inf, 0.002), (3, 0.12, 0.001)])
def test_prox_reference_qp_equals_nested_one_dimensional_searches(seed, tau, kappa):
    """prox_qp (the prox as an Eq. (1) instance with diagonal risk, through the IPM) against prox_nested (the
    definition through one-dimensional golden-section / bisection searches only) on random points v."""
    from oracle import prox_ref
    inst = gen.make_instance("prox", seed, 14, 3, 1, hi_fixed=0.2, tau_fixed=tau if np.isfinite(tau) else None,
                             excl_frac=0.15, kappa_fixed=kappa)
    acc = _acc(inst)                                   # (the generator floors tau so that the exclusions can be sold)
    rng = np.random.default_rng(100 + seed)
    rho = 100.0 * acc.gamma * acc.d
    v = acc.w0 + rng.normal(0.0, 0.08, acc.N)
    r = prox_ref.prox_qp(acc, v, rho, witness=inst.witness[0])
    assert r["status"] == "optimal"
    z_nested = prox_ref.prox_nested(acc, v, rho)
    assert abs(z_nested.sum() - 1.0) < 1e-7
    assert np.max(np.abs(r["w"] - z_nested)) < 2e-7
    # and the answer carries a KKT certificate for the prox problem itself
    _certify(prox_ref.prox_problem(acc, v, rho), r)


def test_prox_reference_box_and_budget_only_is_the_capped_simplex_projection():
    """rho = 1, no cap, no penalty: the prox of the indicator of {1'z = 1, 0 <= z <= u} is the Euclidean projection."""
    from oracle import prox_ref
    inst = gen.make_instance("proxproj", 7, 40, 3, 1, hi_fixed=0.06, gamma_fixed=1.0)
    acc = _acc(inst)
    acc.tau = np.inf
    v = np.random.default_rng(7).normal(0.02, 0.05, acc.N)
    r = prox_ref.prox_qp(acc, v, np.ones(acc.N), witness=inst.witness[0])
    assert np.max(np.abs(r["w"] - closed_form.capped_simplex_projection(v, 0.06))) < 1e-8
