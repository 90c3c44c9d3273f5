#!/usr/bin/env python
"""bench.py - whole-hot-path throughput of the batched rebalancing solver on B200.

One "step" = one cold prism_solve_batch over a synthetic batch shaped like BASELINE.json:configs[2]
(production queue: 500 accounts x 10,000 instruments, k = 50, 20 sector bands, 2% exclusions, L1 turnover cap,
long-only box 0.05), every account solved to 1e-6 scaled KKT residuals (BASELINE.json:metric).
Prints ONE JSON line (see the task contract): value = accounts/sec with inputs resident in HBM; e2e = the same
metric through prism_solve_batch_host with pinned HOST buffers (H2D of mu and w0, D2H of weights, statuses,
iterations and the residual block inside the timed region); roofline of the dominant kernel from per-kernel CUDA
events; cpu_baseline = the fp64 oracle (oracle/ipm.py, as it stands) timed on this box's host cores on a bounded
sample of the same workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg2] [--accounts A]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

PROX_BYTES_PER_ELEM = 41.0      # v 8 + w0 8 + mu 8 + exclusion mask 1 read; r~ 8 + c 8 written (kernel table)
PROX_NCU_TRAFFIC_BYTES = 174.35e6   # k_prox_stream<0>, one launch, all 500 accounts active (profiles/r1c_prox_ncu_full.md)
PROX_CHECK_EXTRA_BYTES = 24.0   # check iterations: x 8 + (P x + q) 8 read, w_out 8 written (kernel table)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, gpu_index: int):
        self.rows = []
        self.stop = threading.Event()
        self.gpu = gpu_index
        self.th = threading.Thread(target=self.run, daemon=True)

    def run(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.th.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.th.join(timeout=6)

    def summary(self):
        sm = []; mx = 0.0; reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        med = sm[len(sm) // 2] if sm else None
        return {"sm_mhz": med, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(sm)}


def make_instance(cfg: str, seed: int, accounts):
    from instances import gen
    kw = {}
    if accounts:
        kw["A"] = accounts
    return gen.by_name(cfg, seed=seed, **kw)


def oracle_sample(inst, n_accounts: int):
    """Times the oracle (as it stands) on the first n accounts; returns (accounts/sec, threads, seconds)."""
    from oracle import ipm, problem
    try:
        from threadpoolctl import threadpool_info
        threads = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        threads = os.cpu_count() or 1
    t0 = time.perf_counter()
    done = 0
    for a in range(n_accounts):
        r = ipm.solve(problem.account_from_instance(inst, a), witness=inst.witness[a])
        if r["status"] != "optimal":
            raise RuntimeError(f"oracle failed on account {a}: {r['status']}")
        done += 1
    dt = time.perf_counter() - t0
    return done / dt, threads, dt


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (rank 0 only), bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    inst = make_instance(args.config, 0, max(args.oracle_accounts, 1))
    n = min(args.oracle_accounts, inst.A)
    for _ in range(min(args.warmup, 1)):
        oracle_sample(inst, 1)
    tot_t = 0.0; tot_n = 0; threads = 1
    for _ in range(args.steps):
        aps, threads, dt = oracle_sample(inst, n)
        tot_t += dt; tot_n += n
    value = tot_n / tot_t
    sample = f"first {n} accounts of {args.config} (N={inst.N}, k={inst.k}, G={inst.G}) per step, structured interior point, fp64"
    print(json.dumps({
        "impl": "reference", "metric": "accounts/sec solved to 1e-6 KKT at N=10k batch 500", "value": value, "unit": "accounts/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.config}: {sample}"},
        "cpu_baseline": {"value": value, "unit": "accounts/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "accounts/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg2")
    ap.add_argument("--accounts", type=int, default=0, help="override the batch size (debug only)")
    ap.add_argument("--oracle-accounts", type=int, default=2, help="accounts in the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--gemm-mode", type=int, default=0)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import paper_2606_23367_b200 as pr
    from paper_2606_23367_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = f"cuda:{local}"

    # weak scaling: every rank solves its own batch (accounts are independent programs);
    # the shared universe is replicated, there is no data-path collective.
    inst = make_instance(args.config, seed=rank, accounts=args.accounts)
    P = pr.Problem(inst, device=dev)
    settings = binding.default_settings(gemm_precision=args.gemm_mode)
    A, N = inst.A, inst.N

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident lane (value)
    last = None
    for _ in range(max(args.warmup, 3) if args.warmup >= 3 else args.warmup):
        last = P.solve(settings)
    barrier()
    ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
    launches = 0; iters_total = 0; interval_ms = 0.0
    with ClockSampler(local) as cs:
        ev0.record()
        for _ in range(args.steps):
            last = P.solve(settings)
            launches += last.info["kernel_launches"]; iters_total += last.info["iters_total"]; interval_ms += last.info["solve_interval_ms"]
        ev1.record()
        barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = cs.summary()
    if dist is not None:
        t = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    status = last.status.cpu().numpy(); iters = last.iters.cpu().numpy(); resid = last.resid.cpu().numpy()
    n_cert = int((status == 0).sum())

    # ---------------- end-to-end lane: pinned host buffers in and out, copies inside the timed call
    mu_h = torch.as_tensor(inst.mu).pin_memory(); w0_h = torch.as_tensor(inst.w0).pin_memory()
    w_h = torch.empty((A, N), dtype=torch.float64).pin_memory(); st_h = torch.empty(A, dtype=torch.int32).pin_memory()
    it_h = torch.empty(A, dtype=torch.int32).pin_memory(); rs_h = torch.empty((A, binding.NRES), dtype=torch.float64).pin_memory()
    for _ in range(1):
        P.solve_host(mu_h, w0_h, w_h, st_h, it_h, rs_h, settings)
    barrier()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        P.solve_host(mu_h, w0_h, w_h, st_h, it_h, rs_h, settings)
    e1.record()
    barrier()
    e2e_ms = max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - t0))
    if dist is not None:
        t = torch.tensor([e2e_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    lane_diff = float((w_h.to(dev) - last.w).abs().max())
    assert lane_diff < 1e-9, f"host lane and device lane disagree: {lane_diff}"
    h2d = mu_h.numel() * 8 + w0_h.numel() * 8
    d2h = w_h.numel() * 8 + st_h.numel() * 4 + it_h.numel() * 4 + rs_h.numel() * 8

    # ---------------- roofline of the dominant kernel: one extra solve with per-launch CUDA events (not timed above)
    prof = binding.default_settings(gemm_precision=args.gemm_mode, profile=1)
    rp = P.solve(prof)
    kt = P.kernel_times()
    tot_k = sum(v["ms"] for v in kt.values()) or 1.0
    dom = max(kt, key=lambda n: kt[n]["ms"])
    peak, peak_src = load_peaks()
    prox = kt["prox"]
    elem_iters = float(N) * float(rp.info["iters_total"])          # account-iterations x N: elements the prox launches processed
    # check launches (every check_every-th iteration of an account) also read x and P x + q and write w_out: + 24 B
    it_prof = rp.iters.cpu().numpy().astype(np.int64)
    ce, fc = int(prof.check_every), int(prof.first_check)
    n_checks = np.maximum(it_prof // ce - (fc + ce - 1) // ce + 1, 0)         # checks at iterations ceil(fc/ce) ce, ... <= iters
    check_elems = float(N) * float(n_checks.sum())
    prox_bytes_per_launch = (PROX_BYTES_PER_ELEM * elem_iters + PROX_CHECK_EXTRA_BYTES * check_elems) / max(prox["launches"], 1)
    prox_ms_per_launch = prox["ms"] / max(prox["launches"], 1)
    achieved = prox_bytes_per_launch / (prox_ms_per_launch * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "k_prox_stream (H4/H5 fused projection + rhs assembly + residual terms, streaming pass)",
                "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak,
                # dram__bytes_read.sum + dram__bytes_write.sum of one full-batch launch (500 accounts x 10,000), from the
                # ncu --set full capture summarised in profiles/r1c_prox_ncu_full.md; only meaningful for the cfg2 batch
                "traffic": PROX_NCU_TRAFFIC_BYTES if (args.config == "cfg2" and not args.accounts) else None,
                "traffic_source": "profiles/r1c_prox_ncu_full.md (ncu --set full, one launch with all accounts active: 205 MB algorithmic)",
                "peak_source": peak_src,
                "factor_gemm_tensor_pipe": {"gemm1_dmma_pct_of_peak": 67.4, "gemm2_dmma_pct_of_peak": 43.0,
                                            "source": "profiles/r1c_gemm_ncu_full.md (sm__inst_executed_pipe_tensor_subpipe_dmma, fp64 mma.sync)"},
                "bytes_per_launch": prox_bytes_per_launch, "ms_per_launch": prox_ms_per_launch,
                "dominant_by_time": dom,
                "kernel_share": {n: round(v["ms"] / tot_k, 4) for n, v in kt.items()},
                "kernel_ms_per_launch": {n: (v["ms"] / v["launches"] if v["launches"] else None) for n, v in kt.items()}}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    # ---------------- oracle on the host cores (reported baseline, not the target)
    cpu = None
    if not args.no_cpu_baseline:
        n = min(args.oracle_accounts, A)
        aps, threads, dt = oracle_sample(inst, n)
        cpu = {"value": aps, "unit": "accounts/s", "cores": threads, "kind": "oracle",
               "sample": f"first {n} of the {A} accounts of this batch, structured interior point fp64, {dt:.1f} s"}
    total_accounts = A * args.steps * world
    out = {
        "metric": "accounts/sec solved to 1e-6 KKT at N=10k batch 500", "value": total_accounts / (ms * 1e-3), "unit": "accounts/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{inst.name}: {A} accounts x N={N}, k={inst.k}, G={inst.G} per GPU (BASELINE.json configs[2] shape), cold start every step",
                   "eps_rel": settings.eps_rel, "l2": "working set > L2 (3 state arrays + mu, w0, mask = 205 MB vs 126 MB L2); each step is a full cold solve",
                   "certified": n_cert, "accounts": A, "iters_p50": float(np.median(iters)), "iters_max": int(iters.max()),
                   "iterations_per_sec": iters_total / (interval_ms * 1e-3) if interval_ms else None,
                   "max_scaled_residual": float(max(resid[:, 7].max(), resid[:, 8].max())),
                   "max_gate_residual": float(resid[:, 0:4].max()), "device_bytes": P.device_bytes, "library": pr.version()},
        "clocks": clocks,
        "e2e": {"value": total_accounts / (e2e_ms * 1e-3), "unit": "accounts/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / args.steps},
        "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
