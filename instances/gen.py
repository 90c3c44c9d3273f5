"""Seeded synthetic instance generator for the PRISM batched rebalancing workload.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2606_23367_b200/`).  It holds no solver arithmetic: it draws
problem data for Eq. (1) of the paper (Section 4.2) in the
concretisation of SURVEY.md 8.0 and `BASELINE.json:configs[0..4]`, and repairs
randomly drawn instances so that they are strictly feasible (SURVEY.md 8(c)
readings R7, R9, R20; Slater premise PAPER.md:126).

Layout of every per-account array: account-major, i.e. shape (A, N) with the N
assets of one account contiguous (C order).  Shared arrays: B (N, k), f (k,),
d (N,), group_id (N,) uint8.

Draw order (reading R23): numpy.random.Generator(PCG64(seed)); shared data
B, f, d, group_id first; then per account a = 0..A-1 in order: mu, gamma, w0,
tau, hi, exclusions, benchmark / lots / caps.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

# constraint-set bit flags (mirror include/prism.h; plain integers, no arithmetic)
F_BUDGET = 1
F_BOX = 2
F_EXCLUSION = 4
F_TURNOVER_CAP = 8
F_TURNOVER_PENALTY = 16
F_GROUP_BANDS = 32
F_TAX_LOTS = 64
F_BUY_COST = 128
F_BENCHMARK_SHIFT = 256

MAX_LOTS = 4


@dataclass
class Instance:
    """One batch W = {P_a : a = 1..A} of Eq. (1) instances over a shared universe."""

    name: str
    seed: int
    N: int
    k: int
    A: int
    G: int
    flags: int
    # shared universe
    B: np.ndarray                 # (N, k) float64 (values exactly representable in fp32 when b_fp32)
    f: np.ndarray                 # (k,)
    d: np.ndarray                 # (N,)
    group_id: Optional[np.ndarray]  # (N,) uint8 or None
    d_t: Optional[np.ndarray]     # (N,) turnover scaling D_t, None => identity
    b_fp32: bool
    # per account
    mu: np.ndarray                # (A, N)
    gamma: np.ndarray             # (A,)
    w0: np.ndarray                # (A, N)
    w_b: Optional[np.ndarray]     # (A, N) benchmark in the risk term, None => 0
    lo: np.ndarray                # (A,) scalar lower bound per account
    hi: np.ndarray                # (A,) scalar upper bound per account (used when hi_full is None)
    hi_full: Optional[np.ndarray]  # (A, N) per-asset caps or None
    excl: Optional[np.ndarray]    # (A, N) uint8, 1 => w_i = 0
    tau: np.ndarray               # (A,)  (+inf => no cap)
    kappa: np.ndarray             # (A,)  L1 transition penalty weight (0 => none)
    band_lo: Optional[np.ndarray]  # (A, G)
    band_hi: Optional[np.ndarray]  # (A, G)
    c_buy: np.ndarray             # (A,)
    lot_slope: Optional[np.ndarray]  # (A, N, MAX_LOTS) ascending within an asset
    lot_width: Optional[np.ndarray]  # (A, N, MAX_LOTS) sums to w0 over the asset's lots
    lot_count: Optional[np.ndarray]  # (A, N) uint8 in 0..MAX_LOTS (0 => no lots on that asset)
    # generator bookkeeping
    witness: np.ndarray = field(default=None)   # (A, N) strictly feasible point
    tau_drawn: np.ndarray = field(default=None)
    n_tau_floored: int = 0
    n_band_widened: int = 0

    def bounds(self, a: int):
        """Effective per-asset (lo, hi) of account a with exclusions folded in."""
        lo = np.full(self.N, float(self.lo[a]))
        hi = self.hi_full[a].copy() if self.hi_full is not None else np.full(self.N, float(self.hi[a]))
        if self.excl is not None:
            m = self.excl[a] != 0
            lo[m] = 0.0
            hi[m] = 0.0
        return lo, hi

    def subset(self, idx) -> "Instance":
        """The same universe restricted to the accounts in idx (a view-free copy)."""
        idx = np.asarray(idx, dtype=np.int64)
        kw = {}
        for fl in dataclasses.fields(self):
            v = getattr(self, fl.name)
            if isinstance(v, np.ndarray) and fl.name not in ("B", "f", "d", "group_id", "d_t") and v.shape[0] == self.A:
                kw[fl.name] = np.ascontiguousarray(v[idx])
            else:
                kw[fl.name] = v
        kw["A"] = len(idx)
        return Instance(**kw)


def _dirichlet_rows(rng, alpha: float, N: int) -> np.ndarray:
    g = rng.standard_gamma(alpha, size=N)
    s = g.sum()
    return g / s


def _witness(w0, lo, hi, group_id, G):
    """Strictly feasible point near w0 (reading R7): clip to the box, then hand the
    freed weight pro-rata to the remaining headroom, same group first."""
    w = np.minimum(np.maximum(w0, lo), hi)
    head = hi - w
    if G > 0:
        for g in range(G):
            m = group_id == g
            deficit = w0[m].sum() - w[m].sum()
            hs = head[m].sum()
            if deficit > 0 and hs > 0:
                frac = min(1.0, deficit / hs) * 0.999999
                w[m] += frac * head[m]
        head = hi - w
    deficit = 1.0 - w.sum()
    if deficit > 0:
        hs = head.sum()
        assert hs > deficit * (1.0 + 1e-9), "Slater premise violated: not enough headroom (PAPER.md:126)"
        w = w + (deficit / hs) * head
    elif deficit < 0:
        room = w - lo
        rs = room.sum()
        assert rs > -deficit * (1.0 + 1e-9)
        w = w + (deficit / rs) * room
    return w


def _finish(inst: Instance, tau_margin: float = 1.25, band_pad: float = 0.1) -> Instance:
    """Feasibility witness, tau-floor (R7), band-floor (R9), Slater assert (R20)."""
    A, N, G = inst.A, inst.N, inst.G
    inst.witness = np.empty((A, N))
    inst.tau_drawn = inst.tau.copy()
    dt = inst.d_t if inst.d_t is not None else np.ones(N)
    for a in range(A):
        lo, hi = inst.bounds(a)
        assert hi.sum() > 1.0 + 1e-6, "Slater: sum of upper bounds must exceed 1 (PAPER.md:126)"
        assert lo.sum() < 1.0 - 1e-6
        w = _witness(inst.w0[a], lo, hi, inst.group_id, G)
        inst.witness[a] = w
        need = float(np.sum(dt * np.abs(w - inst.w0[a])))
        if np.isfinite(inst.tau[a]) and inst.tau[a] < tau_margin * need:
            inst.tau[a] = tau_margin * need
            inst.n_tau_floored += 1
        if G > 0:
            gs = np.bincount(inst.group_id, weights=w, minlength=G)
            hw = 0.5 * (inst.band_hi[a] - inst.band_lo[a])
            new_lo = np.minimum(inst.band_lo[a], gs - band_pad * hw)
            new_hi = np.maximum(inst.band_hi[a], gs + band_pad * hw)
            if np.any(new_lo != inst.band_lo[a]) or np.any(new_hi != inst.band_hi[a]):
                inst.n_band_widened += 1
            inst.band_lo[a], inst.band_hi[a] = new_lo, new_hi
    return inst


def make_instance(name: str, seed: int, N: int, k: int, A: int, *,
                  gamma_range=(0.5, 5.0), gamma_fixed=None,
                  w0_alpha=1.0,
                  hi_range=None, hi_fixed=None,
                  tau_range=None, tau_fixed=None,
                  excl_frac=0.0,
                  G=0, band_half=0.05,
                  kappa_fixed=0.0,
                  lots=False, tax_rate=0.20, c_buy=0.0,
                  cap_frac=0.0, cap_range=(0.0, 0.01),
                  b_fp32=False,
                  benchmark_in_risk=False) -> Instance:
    """General recipe; the five configs below are calls of this with BASELINE.json's numbers."""
    rng = np.random.Generator(np.random.PCG64(seed))
    # shared universe (R4)
    B = rng.standard_normal((N, k)) / np.sqrt(k)
    if b_fp32:
        B = B.astype(np.float32).astype(np.float64)      # R11: stored fp32, both sides see the same values
    f = rng.uniform(0.01, 0.04, size=k)
    d = rng.uniform(0.001, 0.01, size=N)
    group_id = rng.integers(0, G, size=N).astype(np.uint8) if G > 0 else None

    mu = np.empty((A, N)); gamma = np.empty(A); w0 = np.empty((A, N))
    tau = np.full(A, np.inf); hi = np.ones(A); lo = np.zeros(A)
    excl = np.zeros((A, N), dtype=np.uint8) if excl_frac > 0 else None
    band_lo = np.empty((A, G)) if G > 0 else None
    band_hi = np.empty((A, G)) if G > 0 else None
    w_b = np.empty((A, N)) if benchmark_in_risk else None
    hi_full = np.ones((A, N)) if cap_frac > 0 else None
    lot_slope = np.zeros((A, N, MAX_LOTS)) if lots else None
    lot_width = np.zeros((A, N, MAX_LOTS)) if lots else None
    lot_count = np.zeros((A, N), dtype=np.uint8) if lots else None
    n_excl = int(round(excl_frac * N))
    n_cap = int(round(cap_frac * N))

    for a in range(A):
        mu[a] = 0.05 + 0.02 * rng.standard_normal(N)                                  # R3
        gamma[a] = gamma_fixed if gamma_fixed is not None else rng.uniform(*gamma_range)
        w0[a] = _dirichlet_rows(rng, w0_alpha, N)                                       # R5
        if tau_fixed is not None:
            tau[a] = tau_fixed
        elif tau_range is not None:
            tau[a] = rng.uniform(*tau_range)
        if hi_fixed is not None:
            hi[a] = hi_fixed
        elif hi_range is not None:
            hi[a] = rng.uniform(*hi_range)
        if n_excl > 0:
            excl[a, rng.choice(N, size=n_excl, replace=False)] = 1                     # R8
        if G > 0:                                                                      # R9
            wb = _dirichlet_rows(rng, 1.0, N)
            bench = np.bincount(group_id, weights=wb, minlength=G)
            band_lo[a] = bench - band_half
            band_hi[a] = bench + band_half
            if benchmark_in_risk:
                w_b[a] = wb
        elif benchmark_in_risk:
            w_b[a] = _dirichlet_rows(rng, 1.0, N)
        if lots:                                                                       # R10
            L = rng.integers(1, MAX_LOTS + 1, size=N)
            frac = rng.standard_gamma(1.0, size=(N, MAX_LOTS))
            ratio = np.exp(0.3 * rng.standard_normal((N, MAX_LOTS)))
            live = np.arange(MAX_LOTS)[None, :] < L[:, None]
            frac = np.where(live, frac, 0.0)
            frac /= frac.sum(axis=1, keepdims=True)
            slope = np.where(live, tax_rate * np.maximum(1.0 - ratio, 0.0), np.inf)
            order = np.argsort(slope, axis=1, kind="stable")
            slope = np.take_along_axis(slope, order, axis=1)
            frac = np.take_along_axis(frac, order, axis=1)
            slope = np.where(np.isfinite(slope), slope, 0.0)
            lot_slope[a] = slope
            lot_width[a] = frac * w0[a][:, None]
            lot_count[a] = L.astype(np.uint8)
        if n_cap > 0:
            ci = rng.choice(N, size=n_cap, replace=False)
            hi_full[a, ci] = rng.uniform(*cap_range, size=n_cap)

    flags = F_BUDGET | F_BOX
    if excl is not None: flags |= F_EXCLUSION
    if np.any(np.isfinite(tau)): flags |= F_TURNOVER_CAP
    if kappa_fixed > 0: flags |= F_TURNOVER_PENALTY
    if G > 0: flags |= F_GROUP_BANDS
    if lots: flags |= F_TAX_LOTS
    if c_buy > 0: flags |= F_BUY_COST
    if benchmark_in_risk: flags |= F_BENCHMARK_SHIFT

    inst = Instance(name=name, seed=seed, N=N, k=k, A=A, G=G, flags=flags,
                    B=B, f=f, d=d, group_id=group_id, d_t=None, b_fp32=b_fp32,
                    mu=mu, gamma=gamma, w0=w0, w_b=w_b, lo=lo, hi=hi, hi_full=hi_full,
                    excl=excl, tau=tau, kappa=np.full(A, float(kappa_fixed)),
                    band_lo=band_lo, band_hi=band_hi, c_buy=np.full(A, float(c_buy)),
                    lot_slope=lot_slope, lot_width=lot_width, lot_count=lot_count)
    return _finish(inst)


# ----------------------------------------------------------------------------------------------
# BASELINE.json:configs[0..4] and scaled-down replicas for parity tests
# ----------------------------------------------------------------------------------------------

def config0(seed=0, N=100, k=10):
    """configs[0]: single account, budget + box [0,0.10] + ||w-w0||_1 <= 0.20, gamma = 1."""
    return make_instance("cfg0_single", seed, N, k, 1, gamma_fixed=1.0, hi_fixed=0.10, tau_fixed=0.20)


def config1(seed=0, N=2000, k=30, A=100):
    """configs[1]: 100 accounts, N=2,000, k=30, tau~U[.05,.3], hi~U[.02,.1], 5% exclusions."""
    return make_instance("cfg1_batch", seed, N, k, A, tau_range=(0.05, 0.3), hi_range=(0.02, 0.1),
                         excl_frac=0.05)


def config2(seed=0, N=10000, k=50, A=500, G=20, band_half=0.05):
    """configs[2]: production queue, 500 x 10,000, k=50, 20 sector bands, 2% exclusions, hi=0.05."""
    return make_instance("cfg2_queue", seed, N, k, A, tau_range=(0.05, 0.25), hi_fixed=0.05,
                         excl_frac=0.02, G=G, band_half=band_half)


def config3(seed=0, N=10000, k=50, A=200):
    """configs[3]: tax-aware batch, lots (1-4 per asset), buy cost 5 bp, caps on 10%, tau = 0.15."""
    return make_instance("cfg3_tax", seed, N, k, A, tau_fixed=0.15, hi_fixed=1.0, lots=True,
                         c_buy=5e-4, cap_frac=0.10, cap_range=(0.0, 0.01))


def config4(seed=0, N=384800, k=100, A=32, hi=0.001):
    """configs[4]: wide universe, fp32 loadings, hi = 0.001, 1% exclusions, tau = 0.10, Dir(0.1)."""
    return make_instance("cfg4_wide", seed, N, k, A, tau_fixed=0.10, hi_fixed=hi, excl_frac=0.01,
                         w0_alpha=0.1, b_fp32=True)


def section9(seed=0, N=481, k=20, A=1, kappa=0.005, cap=0.03):
    """PAPER.md:378 transition objective in 8.0 form (reading R14): gamma=2, f=1, L1 penalty kappa, no cap."""
    inst = make_instance("sec9_transition", seed, N, k, A, gamma_fixed=2.0, hi_fixed=cap, kappa_fixed=kappa)
    inst.f = np.ones(k)
    return inst


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def by_name(name: str, seed: int = 0, **kw) -> Instance:
    table = {"cfg0": config0, "cfg1": config1, "cfg2": config2, "cfg3": config3, "cfg4": config4,
             "sec9": section9}
    return table[name](seed=seed, **kw)
