"""Reject-side pins of the independent checker oracle/kkt_check.py: hand-computed values that a
plausible mistake in the checker (a dropped term, a wrong sign, a lot branch that accepts everything) would miss.
Every expected number below is worked out in the comment next to it, not by calling the checker.  CPU only."""
import numpy as np
import pytest

from oracle import kkt_check, problem


def _account(**kw):
    """Four assets, two groups {0,1} and {2,3}, w0 = 1/4 each, identity-free factor part (B = 0), d = 0.02."""
    base = dict(N=4, B=np.zeros((4, 1)), f=np.ones(1), d=np.full(4, 0.02), mu=np.full(4, 0.05), gamma=2.0,
                w0=np.full(4, 0.25), w_b=None, lo=np.zeros(4), hi=np.full(4, 0.4), dt=np.ones(4), tau=10.0, kappa=0.0,
                c_buy=0.0, group_id=np.array([0, 0, 1, 1]), G=2, band_lo=np.array([0.3, 0.3]), band_hi=np.array([0.6, 0.6]),
                lot_slope=None, lot_width=None, lot_count=None)
    base.update(kw)
    return problem.Account(**base)


# ------------------------------------------------------------------------------------------ feasibility residuals
def test_r_box_upper_and_lower_side():
    acc = _account()
    f = kkt_check.feasibility(acc, np.array([0.41, 0.09, 0.25, 0.25]))       # 0.41 - hi 0.40 = 0.01; sum = 1; groups 0.5 / 0.5
    assert abs(f["r_box"] - 0.01) < 1e-15 and f["r_budget"] < 1e-15 and f["r_exposure"] == 0.0 and f["r_turnover"] == 0.0
    f = kkt_check.feasibility(acc, np.array([-0.02, 0.32, 0.35, 0.35]))      # lo 0 - (-0.02) = 0.02; groups 0.30 / 0.70 -> 0.10
    assert abs(f["r_box"] - 0.02) < 1e-15
    assert abs(f["r_exposure"] - 0.10) < 1e-15                                # 0.70 - band_hi 0.60


def test_r_exposure_upper_and_lower_band():
    acc = _account()
    f = kkt_check.feasibility(acc, np.array([0.35, 0.30, 0.175, 0.175]))     # group 0: 0.65 - 0.60 = 0.05; group 1: 0.35 inside
    assert abs(f["r_exposure"] - 0.05) < 1e-15 and f["r_box"] == 0.0
    acc = _account(band_lo=np.array([0.3, 0.45]))
    f = kkt_check.feasibility(acc, np.array([0.30, 0.30, 0.20, 0.20]))       # group 1: band_lo 0.45 - 0.40 = 0.05
    assert abs(f["r_exposure"] - 0.05) < 1e-15


def test_r_turnover_with_and_without_scaling():
    acc = _account(tau=0.1)
    w = np.array([0.35, 0.15, 0.25, 0.25])                                    # |dw| = 0.1 + 0.1 = 0.2 -> 0.2 - tau 0.1 = 0.1
    f = kkt_check.feasibility(acc, w)
    assert abs(f["r_turnover"] - 0.1) < 1e-15 and f["r_box"] == 0.0 and f["r_exposure"] == 0.0
    acc = _account(tau=0.1, dt=np.array([2.0, 1.0, 1.0, 1.0]))                # D_a: 2 * 0.1 + 0.1 = 0.3 -> 0.2
    assert abs(kkt_check.feasibility(acc, w)["r_turnover"] - 0.2) < 1e-15
    assert kkt_check.feasibility(_account(tau=0.25), w)["r_turnover"] == 0.0  # slack cap: no residual
    assert kkt_check.feasibility(_account(tau=np.inf), w)["r_turnover"] == 0.0


def test_lot_sell_limit_counts_as_box():
    """Sells of an asset with lots are limited to the lots held (R10): w >= w0 - sum of widths."""
    acc = _account(lot_slope=np.tile([0.0, 0.02], (4, 1)), lot_width=np.tile([0.05, 0.05], (4, 1)), lot_count=np.full(4, 2))
    f = kkt_check.feasibility(acc, np.array([0.12, 0.38, 0.25, 0.25]))       # floor 0.25 - 0.10 = 0.15; 0.15 - 0.12 = 0.03
    assert abs(f["r_box"] - 0.03) < 1e-15


# ------------------------------------------------------------------------------------------ the lot subdifferential
def _lots_account():
    # one asset of interest (index 0): w0 = 0.30, lots (width 0.10 at slope 0.00), (width 0.10 at slope 0.02); c_buy = 0.001
    return _account(w0=np.array([0.30, 0.30, 0.20, 0.20]), c_buy=0.001, G=0, group_id=None, band_lo=None, band_hi=None,
                    lot_slope=np.tile([0.0, 0.02], (4, 1)), lot_width=np.tile([0.10, 0.10], (4, 1)), lot_count=np.full(4, 2))


@pytest.mark.parametrize("w_first,lo,hi", [
    (0.35, 0.001, 0.001),          # buying: d phi / dw = c_buy
    (0.30, -0.0, 0.001),           # on the kink: [-slope of the first lot, c_buy]
    (0.25, -0.0, -0.0),            # selling 0.05, inside lot 1 (slope 0)
    (0.20, -0.02, -0.0),           # selling 0.10: the breakpoint between the lots -> [-0.02, -0.00]
    (0.15, -0.02, -0.02),          # selling 0.15, inside lot 2 (slope 0.02)
    (0.10, -np.inf, -0.02),        # every lot sold: no further selling possible
])
def test_phi_interval_of_a_two_lot_asset(w_first, lo, hi):
    acc = _lots_account()
    w = acc.w0.copy(); w[0] = w_first
    plo, phi = kkt_check._phi_interval(acc, w, 1e-9)
    assert plo[0] == lo and phi[0] == hi, (plo[0], phi[0])


def test_wrong_lot_answer_is_rejected_with_the_hand_computed_distance():
    """Stationarity of asset 0 when it sells INSIDE lot 2 needs g_0 = +slope_2 = 0.02 exactly (S_0 = {-0.02}); with
    multipliers that are right for a sale inside lot 1 (g_0 = 0) the distance is 0.02 - a checker whose lot branch
    returned [-inf, c_buy] for every lot asset would report 0."""
    acc = _lots_account()
    w = np.array([0.15, 0.45, 0.20, 0.20])            # asset 0 sells 0.15 (lot 2), asset 1 buys 0.15
    # g_i = gamma d_i w_i - mu_i + nu  (B = 0): choose nu so that g_0 = 0:  nu = mu - gamma d w_0 = 0.05 - 2*0.02*0.15 = 0.044
    nu = 0.05 - 2.0 * 0.02 * 0.15
    k = kkt_check.kkt(acc, w, dict(nu=nu, theta=0.0, lam_hi=np.zeros(0), lam_lo=np.zeros(0)), delta=1e-9)
    # asset 0: S = {-0.02}, -g_0 = 0 -> distance 0.02.  asset 1 (buying): S = {c_buy} = {0.001}, g_1 = 2*0.02*0.45 - 0.05 + 0.044
    # = 0.012 -> -g_1 = -0.012, distance 0.013.  assets 2, 3 (w = w0 = 0.20, on the kink): S = [-0, 0.001], g = 0.008 - 0.05 + 0.044
    # = 0.002 -> -g = -0.002, distance 0.002.  r_stat = max = 0.02, attained at asset 0.
    assert abs(k["r_stat"] - 0.02) < 1e-15 and k["worst"] == 0
    # the same point with the sale inside lot 1 (0.05) IS stationary for asset 0 with that g_0 = 0 convention:
    w1 = np.array([0.25, 0.35, 0.20, 0.20])
    nu1 = 0.05 - 2.0 * 0.02 * 0.25
    k1 = kkt_check.kkt(acc, w1, dict(nu=nu1, theta=0.0, lam_hi=np.zeros(0), lam_lo=np.zeros(0)), delta=1e-9)
    # asset 0 distance 0; asset 1: g_1 = 0.014 - 0.05 + 0.04 = 0.004, S = {0.001}, distance 0.005 (largest)
    assert abs(k1["r_stat"] - 0.005) < 1e-15 and k1["worst"] == 1


# ------------------------------------------------------------------------------------------ certificates
def test_r_comp_and_multiplier_signs():
    acc = _account(tau=0.3)
    w = np.array([0.35, 0.15, 0.25, 0.25])                                    # turnover 0.2 (slack 0.1), groups 0.5 / 0.5
    m = dict(nu=0.0, theta=0.5, lam_hi=np.array([0.2, 0.0]), lam_lo=np.array([0.0, 0.1]))
    k = kkt_check.kkt(acc, w, m)
    # theta |turnover - tau| = 0.5 * 0.1 = 0.05; lam_hi_0 |0.5 - 0.6| = 0.02; lam_lo_1 |0.3 - 0.5| = 0.02 -> 0.05
    assert abs(k["r_comp"] - 0.05) < 1e-15 and k["min_multiplier"] == 0.0
    m["lam_lo"] = np.array([0.0, -0.1])
    assert kkt_check.kkt(acc, w, m)["min_multiplier"] == -0.1


def test_certify_free_fails_on_a_feasible_non_optimal_point_and_passes_at_the_optimum():
    """Budget-only optimum of the 2-asset golden case A (tests/golden): w = (0.875, 0.125), nu = 0.0325.  The LP certificate
    must reach 0 there and must NOT reach 0 at a feasible point next to it: at w = (0.8, 0.2) the two stationarity rows
    g_1 + nu = 2*0.01*0.8 - 0.05 + nu and g_2 + nu = 2*0.03*0.2 - 0.04 + nu differ by 0.006, so min_nu max|.| = 0.003."""
    acc = problem.Account(N=2, B=np.zeros((2, 1)), f=np.ones(1), d=np.array([0.01, 0.03]), mu=np.array([0.05, 0.04]), gamma=2.0,
                          w0=np.array([0.5, 0.5]), w_b=None, lo=np.full(2, -5.0), hi=np.full(2, 5.0), dt=np.ones(2), tau=np.inf,
                          kappa=0.0, c_buy=0.0, group_id=None, G=0, band_lo=None, band_hi=None, lot_slope=None, lot_width=None,
                          lot_count=None)
    good = kkt_check.certify_free(acc, np.array([0.875, 0.125]))
    assert good["ok"] and good["r_stat"] < 1e-12 and abs(good["nu"] - 0.0325) < 1e-9
    bad = kkt_check.certify_free(acc, np.array([0.8, 0.2]))
    assert bad["ok"] and abs(bad["r_stat"] - 0.003) < 1e-9


def test_distance_bound_value():
    acc = _account()                                                          # m = gamma min d = 2 * 0.02 = 0.04
    assert abs(kkt_check.distance_bound(acc, 2e-10) - np.sqrt(2 * 2e-10 / 0.04)) < 1e-18      # = 1e-4
    assert abs(kkt_check.distance_bound(acc, 2e-10) - 1e-4) < 1e-15
    assert kkt_check.distance_bound(acc, -1.0) == 0.0
