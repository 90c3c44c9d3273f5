#!/usr/bin/env python
"""bench.py - whole-hot-path throughput of the batched rebalancing solver on B200.

One "step" = one cold prism_solve_batch over a synthetic batch shaped like BASELINE.json:configs[2]
(production queue: 500 accounts x 10,000 instruments, k = 50, 20 sector bands, 2% exclusions, L1 turnover cap,
long-only box 0.05), every account solved to 1e-6 scaled KKT residuals (BASELINE.json:metric).
Prints ONE JSON line (see the task contract): value = accounts/sec with inputs resident in HBM; e2e = the same
metric through prism_solve_batch_host with pinned HOST buffers (H2D of mu and w0, D2H of weights, statuses,
iterations and the residual block inside the timed region); roofline of the kernel class that dominates the solve
(per-launch CUDA events of a separate profiled solve; GEMM fractions against an fp64 yardstick measured in the same
run); `extra`: the same solve on the other configured shapes and the N sweep; cpu_baseline = the fp64 oracle
(oracle/ipm.py, as it stands) on this box's host cores, accounts in parallel processes, on a random sample.

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


def _oracle_one(args):
    """Worker process: one account through the oracle as it stands, one BLAS thread (the parallelism is over accounts)."""
    cfg, seed, A, a = args
    try:
        from threadpoolctl import threadpool_limits
        ctx = threadpool_limits(limits=1)
    except Exception:
        ctx = None
    from instances import gen
    from oracle import ipm, problem
    global _ORACLE_INST
    key = (cfg, seed, A)
    if globals().get("_ORACLE_KEY") != key:
        globals()["_ORACLE_INST"] = gen.by_name(cfg, seed=seed, **({"A": A} if A else {}))
        globals()["_ORACLE_KEY"] = key
    inst = globals()["_ORACLE_INST"]
    t0 = time.perf_counter()
    r = ipm.solve(problem.account_from_instance(inst, a), witness=inst.witness[a])
    return a, r["status"], time.perf_counter() - t0


def _oracle_init():
    """One BLAS thread per worker: environment first (numpy is not loaded yet in a spawned worker), then threadpoolctl."""
    for v in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS"):
        os.environ[v] = "1"
    try:
        import numpy  # noqa: F401
        from threadpoolctl import threadpool_limits
        globals()["_ORACLE_LIMIT"] = threadpool_limits(limits=1)
    except Exception:
        pass


class OraclePool:
    """The fp64 oracle (oracle/ipm.py, untuned) on the host cores: accounts in parallel worker processes, one account
    per process at a time, one BLAS thread each.  cores = number of worker processes."""

    def __init__(self, cfg, seed, accounts, procs=None):
        import multiprocessing as mp
        self.cfg, self.seed, self.A = cfg, seed, accounts
        self.procs = procs or max(1, min(os.cpu_count() or 1, 32))
        self.pool = mp.get_context("spawn").Pool(self.procs, initializer=_oracle_init)

    def run(self, account_ids):
        """Solves the listed accounts; returns (accounts/sec, seconds)."""
        t0 = time.perf_counter()
        out = self.pool.map(_oracle_one, [(self.cfg, self.seed, self.A, int(a)) for a in account_ids], chunksize=1)
        dt = time.perf_counter() - t0
        bad = [(a, st) for a, st, _ in out if st != "optimal"]
        if bad:
            raise RuntimeError(f"oracle failed on accounts {bad[:4]}")
        return len(account_ids) / dt, dt

    def close(self):
        self.pool.close(); self.pool.join()


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (rank 0 only).  Each step solves a bounded random sample of
    the workload's accounts, sized after the warm-up step so that the whole run ends within a few minutes."""
    import numpy as np
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    A_full = args.accounts or {"cfg0": 1, "cfg1": 100, "cfg2": 500, "cfg3": 200, "cfg4": 32}.get(cfg, 100)
    pool = OraclePool(cfg, 0, args.accounts)
    rng = np.random.default_rng(0)
    n = min(pool.procs, A_full)
    ids = rng.choice(A_full, size=n, replace=False)
    _, t1 = pool.run(ids)                                         # warm-up step (also builds the instance in every worker)
    _, t1 = pool.run(ids)
    budget = 200.0                                                # seconds for the timed steps
    per_step = max(1, min(n, int(n * budget / max(args.steps * t1, 1e-9))))
    tot_t = 0.0; tot_n = 0
    for _ in range(args.steps):
        ids = rng.choice(A_full, size=per_step, replace=False)
        _, dt = pool.run(ids)
        tot_t += dt; tot_n += per_step
    pool.close()
    value = tot_n / tot_t
    sample = (f"{per_step} randomly chosen accounts of {cfg} per step ({A_full} in the batch), oracle/ipm.py structured interior point "
              f"fp64, one account per worker process, {pool.procs} processes x 1 BLAS thread")
    print(json.dumps({
        "impl": "reference", "metric": "accounts/sec solved to 1e-6 KKT at N=10k batch 500", "value": value, "unit": "accounts/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{cfg}: {sample}"},
        "cpu_baseline": {"value": value, "unit": "accounts/s", "cores": pool.procs, "kind": "oracle", "sample": sample},
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
    ap.add_argument("--oracle-accounts", type=int, default=32, help="accounts in the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the rows for the other configs and the N sweep")
    ap.add_argument("--gemm-precision", type=int, default=3, help="PRISM_GEMM_*: 3 = 3xTF32 tensor path (library default), 0 = fp64 DMMA")
    ap.add_argument("--prox-form", type=int, default=0, help="PRISM_PROX_* (0 = AUTO) for the headline problem object")
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
    torch.cuda.synchronize()
    t_c0 = time.perf_counter()
    P = pr.Problem(inst, device=dev, prox_form=args.prox_form)
    settings = binding.default_settings(gemm_precision=args.gemm_precision)
    first = P.solve(settings)
    torch.cuda.synchronize()
    create_plus_solve_ms = 1e3 * (time.perf_counter() - t_c0)      # upload + prism_problem_create + first cold solve (R17)
    A, N = inst.A, inst.N

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def allmax(x):
        if dist is None:
            return x
        t = torch.tensor([x], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # ---------------- device-resident lane (value): only certified accounts count
    last = first
    for _ in range(max(args.warmup, 3)):
        last = P.solve(settings)
    barrier()
    ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
    launches = 0; iters_total = 0; interval_ms = 0.0; certified = 0
    with ClockSampler(local) as cs:
        ev0.record()
        for _ in range(args.steps):
            last = P.solve(settings)
            launches += last.info["kernel_launches"]; iters_total += last.info["iters_total"]
            interval_ms += last.info["solve_interval_ms"]; certified += last.info["n_certified"]
        ev1.record()
        barrier()
    ms = allmax(ev0.elapsed_time(ev1))
    clocks = cs.summary()
    status = last.status.cpu().numpy(); iters = last.iters.cpu().numpy(); resid = last.resid.cpu().numpy()
    n_cert = int((status == 0).sum())

    # ---------------- end-to-end lane: pinned host buffers in and out, copies inside the timed call
    mu_h = torch.as_tensor(inst.mu).pin_memory(); w0_h = torch.as_tensor(inst.w0).pin_memory()
    w_h = torch.empty((A, N), dtype=torch.float64).pin_memory(); st_h = torch.empty(A, dtype=torch.int32).pin_memory()
    it_h = torch.empty(A, dtype=torch.int32).pin_memory(); rs_h = torch.empty((A, binding.NRES), dtype=torch.float64).pin_memory()
    P.solve_host(mu_h, w0_h, w_h, st_h, it_h, rs_h, settings)
    barrier()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e2e_cert = 0
    e0.record()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        P.solve_host(mu_h, w0_h, w_h, st_h, it_h, rs_h, settings)
        e2e_cert += int((st_h.numpy() == 0).sum())
    e1.record()
    barrier()
    e2e_ms = allmax(max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - t0)))
    lane_diff = float((w_h.to(dev) - last.w).abs().max())
    assert lane_diff < 1e-9, f"host lane and device lane disagree: {lane_diff}"
    h2d = mu_h.numel() * 8 + w0_h.numel() * 8
    d2h = w_h.numel() * 8 + st_h.numel() * 4 + it_h.numel() * 4 + rs_h.numel() * 8

    # ---------------- per-kernel accounting: one extra solve with per-launch CUDA events (not part of the timings above)
    peak, peak_src = load_peaks()
    yard = P.fp64_yardstick()                                      # measured on this device, this run

    def profile(Pq, instq):
        """Per-kernel-class device time of one profiled solve and the algorithmic bytes / flops it stands for."""
        rp = Pq.solve(binding.default_settings(gemm_precision=args.gemm_precision, profile=1))
        kt = Pq.kernel_times()
        tot = sum(v["ms"] for v in kt.values()) or 1.0
        itp = rp.iters.cpu().numpy().astype(np.int64)
        ce, fc = 10, 40                                             # check_every, first_check defaults
        n_checks = np.maximum(itp // ce - (fc + ce - 1) // ce + 1, 0)
        elem_it = float(instq.N) * float(itp.sum()); elem_ck = float(instq.N) * float(n_checks.sum())
        lots = instq.lot_slope is not None
        per = {}
        # H4 (+H5-H7): the fused projection; for the streaming form both of its kernels (k_prox_stream + k_prox_root)
        # lots / caps: the pass reads per asset the cap 8 B, the lot count 1 B and the first slope 8 B (lot rows only for live assets)
        b_prox = (PROX_BYTES_PER_ELEM + (17.0 if lots else 0.0)) * elem_it + PROX_CHECK_EXTRA_BYTES * elem_ck
        b_g2 = 24.0 * elem_it + 24.0 * elem_ck                      # v, c read, v written (+ r~ read, x, Px+q written on checks)
        b_g1 = 8.0 * elem_it                                        # r~ read
        fl = 2.0 * instq.k * elem_it                                # per GEMM
        for name, nbytes, flops in (("prox", b_prox, 0.0), ("gemm2", b_g2, fl), ("gemm1", b_g1, fl)):
            t = kt[name]["ms"] * 1e-3
            if t <= 0:
                continue
            per[name] = {"ms": kt[name]["ms"], "launches": kt[name]["launches"], "share": kt[name]["ms"] / tot,
                         "algorithmic_GBps": nbytes / t / 1e9, "hbm_frac": nbytes / t / 1e9 / peak}
            if flops:
                per[name]["TFLOPs"] = flops / t / 1e12          # contraction flops 2 N k per account-iteration
                if args.gemm_precision in (0, 1):
                    per[name]["frac_of_measured_dmma"] = flops / t / 1e12 / yard["dmma_tflops"]
                else:
                    per[name]["tensor_path"] = "3xTF32 mma.sync m16n8k8 (3 MMAs per product, fp32 accumulate): HBM-bound, see hbm_frac"
        for name in ("solve", "factor", "diag", "other"):
            if kt[name]["ms"] > 0:
                per[name] = {"ms": kt[name]["ms"], "launches": kt[name]["launches"], "share": kt[name]["ms"] / tot}
        dom = max(kt, key=lambda n: kt[n]["ms"])
        return rp, kt, per, dom, tot, b_prox + b_g2 + b_g1

    rp, kt, per, dom, tot_k, step_bytes = profile(P, inst)
    domk = per[dom]
    FORMS = {1: "k_prox_res (cluster-resident form)", 2: "k_prox_stream + k_prox_root (streaming form)", 3: "k_prox (every-asset form)"}
    gk = "_tf32" if args.gemm_precision == 3 else ""
    kernel_names = {"prox": "H4-H7 fused projection: " + FORMS[P.prox_form],
                    "gemm2": f"H3 k_gemm2{gk} (factor GEMM-2 + epilogue)", "gemm1": f"H1 k_gemm1{gk} (split-K factor GEMM-1)"}
    roofline = {"bound": "hbm", "kernel": kernel_names.get(dom, dom), "dominant_by_time": dom,
                "achieved": domk.get("algorithmic_GBps"), "peak": peak, "unit": "GB/s",
                "frac": domk.get("hbm_frac"), "traffic": None,
                "traffic_note": "not measured inside bench.py; ncu dram bytes per launch are in profiles/r2_*.md",
                "peak_source": peak_src,
                "bytes_per_launch": (domk["algorithmic_GBps"] * 1e9 * domk["ms"] * 1e-3 / max(domk["launches"], 1)) if "algorithmic_GBps" in domk else None,
                "ms_per_launch": domk["ms"] / max(domk["launches"], 1),
                "whole_step": {"algorithmic_GBps": step_bytes / (rp.info["solve_interval_ms"] * 1e-3) / 1e9,
                               "hbm_frac": step_bytes / (rp.info["solve_interval_ms"] * 1e-3) / 1e9 / peak,
                               "bytes_per_element_iteration": "prox 41 (+24 on check iterations) + gemm1 8 + gemm2 24 (+24)"},
                "fp64_yardstick_TFLOPs": yard, "gemm_precision": {0: "fp64 DMMA", 1: "fp64 FMA", 2: "fp32 experiment", 3: "3xTF32"}[args.gemm_precision],
                "per_kernel": per}

    def row(name, instq, form=0):
        Pq = pr.Problem(instq, device=dev, prox_form=form)
        Pq.solve(settings)
        r = Pq.solve(settings)
        _, ktq, perq, domq, _, _ = profile(Pq, instq)
        itq = r.iters.cpu().numpy(); stq = r.status.cpu().numpy(); rsq = r.resid.cpu().numpy()
        out = {"config": name, "A": instq.A, "N": instq.N, "k": instq.k, "G": instq.G, "solve_ms": r.info["solve_interval_ms"],
               "accounts_per_s": int((stq == 0).sum()) / (r.info["wall_ms"] * 1e-3), "certified": int((stq == 0).sum()),
               "iters_p50": float(np.median(itq)), "iters_max": int(itq.max()),
               "iterations_per_sec": r.info["iters_total"] / (r.info["solve_interval_ms"] * 1e-3),
               "max_scaled_residual": float(max(rsq[:, 7].max(), rsq[:, 8].max())), "max_gate_residual": float(rsq[:, 0:4].max()),
               "prox_form": FORMS[Pq.prox_form], "dominant_kernel": domq, "kernel_share": {n: round(v["share"], 3) for n, v in perq.items()},
               "launches": int(r.info["kernel_launches"]), "device_bytes": Pq.device_bytes}
        Pq.close()
        return out

    t_sec = time.perf_counter()
    extra = []
    if rank == 0 and not args.no_extra:
        from instances import gen
        for name in ("cfg0", "cfg1", "cfg3", "cfg4"):
            if name != args.config:
                extra.append(row(name, gen.by_name(name, seed=0)))
        for Ns, ks in ((100, 10), (500, 20), (1000, 30), (2000, 30)):       # R24: N sweep, A = 100, configs[1] distributions
            extra.append(row(f"sweep_N{Ns}", gen.config1(seed=0, N=Ns, k=ks, A=100)))
        # NEXT-1: the paper's transition-penalty family (reading R14) on its single-account scale
        # ladder N = 481 x {1, 4, 20, 100, 800} (Table 12): timing rows, parity is the sec9 test case
        for mult in (1, 4, 20, 100, 800):
            extra.append(dict(row(f"sec9_ladder_N{481 * mult}", gen.section9(seed=0, N=481 * mult, k=20, A=1)),
                              note="single account, L1 penalty kappa = 0.005, cap 3%, no turnover cap"))
        if args.config == "cfg2":                                            # the paper's queue framing (Table 8) on the headline batch
            from paper_2606_23367_b200 import queue_layer
            for bs, lanes in ((500, 1), (125, 1), (125, 4)):
                queue_layer.run_queue(inst, batch_size=bs, lanes=lanes, device=dev)          # warm-up (first-touch of the allocations)
                _, recs = queue_layer.run_queue(inst, batch_size=bs, lanes=lanes, deadline_ms=1.5e6, device=dev)
                extra.append(dict(queue_layer.summarise(recs), config=f"queue_cfg2_batches_of_{bs}" + (f"_lanes_{lanes}" if lanes > 1 else ""),
                                  note="NEXT-3 queue layer: consecutive batches incl. prism_problem_create per batch, 1,500 s window; "
                                       "latency = queue start -> result available; paper: 109.5 s total, p50 212 ms per account on its hardware"))
            # a deeper queue: four times the batch (the same accounts, replicated) as four batches of 500 in four lanes -
            # one solve is a chain of short launches that leaves most of the GPU idle, independent batches fill it
            inst4 = inst.subset(list(range(inst.A)) * 4)
            queue_layer.run_queue(inst4, batch_size=inst.A, lanes=4, device=dev)
            _, recs = queue_layer.run_queue(inst4, batch_size=inst.A, lanes=4, deadline_ms=1.5e6, device=dev)
            extra.append(dict(queue_layer.summarise(recs), config=f"queue_4x_cfg2_batches_of_{inst.A}_lanes_4",
                              note="2,000 accounts (the headline batch four times) as four concurrent batches, one host thread and CUDA stream each, "
                                   "incl. prism_problem_create and the read-back of every batch"))
            del inst4
            # the same without the host-side work: four resident problem objects of the headline batch solved at once
            Ps = [binding.Problem(inst, device=dev, prox_form=args.prox_form) for _ in range(4)]
            queue_layer.solve_concurrently(Ps, gemm_precision=args.gemm_precision)
            rs4, ms4 = min((queue_layer.solve_concurrently(Ps, gemm_precision=args.gemm_precision) for _ in range(3)), key=lambda x: x[1])
            extra.append(dict(config="cfg2_four_resident_batches_at_once", A=4 * inst.A, N=inst.N, ms_per_solve=ms4,
                              accounts_per_s=sum(int((r.status == 0).sum()) for r in rs4) / (ms4 * 1e-3),
                              certified=sum(int((r.status == 0).sum()) for r in rs4),
                              note="four problem objects of the headline batch, one host thread and CUDA stream each, wall clock between device "
                                   "synchronisations; the headline value above is ONE batch at a time"))
            for P4 in Ps:
                P4.close()
        if args.config == "cfg2":                                            # configs[3] as four sub-batches of 50 accounts at once
            from paper_2606_23367_b200 import queue_layer, shard
            inst3 = gen.config3(seed=0)
            q = [shard.slice_instance(inst3, a0, a1) for a0, a1 in zip(range(0, inst3.A, 50), range(50, inst3.A + 50, 50))]
            Ps = [binding.Problem(x, device=dev) for x in q]
            queue_layer.solve_concurrently(Ps, gemm_precision=args.gemm_precision)
            rs3, ms3 = min((queue_layer.solve_concurrently(Ps, gemm_precision=args.gemm_precision) for _ in range(3)), key=lambda x: x[1])
            extra.append(dict(config="cfg3_four_sub_batches_at_once", A=inst3.A, N=inst3.N, ms_per_solve=ms3,
                              accounts_per_s=sum(int((r.status == 0).sum()) for r in rs3) / (ms3 * 1e-3),
                              certified=sum(int((r.status == 0).sum()) for r in rs3),
                              note="configs[3] cut into four resident problem objects of 50 accounts, solved at once on four streams (wall clock); "
                                   "the cfg3 row above is the same batch as ONE problem object"))
            for P3 in Ps:
                P3.close()
            del inst3, q
        if args.config == "cfg2":                                            # the other form of the projection on the headline batch
            extra.append(dict(row("cfg2_resident_form", inst, form=binding.PROX_RESIDENT), note="prox_form = PRISM_PROX_RESIDENT"))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    sys.stderr.write(f"[bench] extra rows: {time.perf_counter() - t_sec:.1f} s\n"); t_sec = time.perf_counter()
    # ---------------- oracle on the host cores (reported baseline, not the target)
    cpu = None
    if not args.no_cpu_baseline:
        n = min(args.oracle_accounts, A)
        pool = OraclePool(args.config, rank, args.accounts)
        ids = np.random.default_rng(0).choice(A, size=n, replace=False)
        pool.run(ids[:min(len(ids), pool.procs)])                            # builds the instance in every worker (untimed)
        aps, dt = pool.run(ids)
        pool.close()
        cpu = {"value": aps, "unit": "accounts/s", "cores": pool.procs, "kind": "oracle",
               "sample": f"{n} randomly chosen accounts of the {A} of this batch, oracle/ipm.py structured interior point fp64, "
                         f"one account per worker process ({pool.procs} processes x 1 BLAS thread), {dt:.1f} s"}
    sys.stderr.write(f"[bench] cpu baseline: {time.perf_counter() - t_sec:.1f} s\n")
    out = {
        "metric": "accounts/sec solved to 1e-6 KKT at N=10k batch 500", "value": certified * world / (ms * 1e-3), "unit": "accounts/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{inst.name}: {A} accounts x N={N}, k={inst.k}, G={inst.G} per GPU (BASELINE.json configs[2] shape), cold start every step",
                   "eps_rel": settings.eps_rel, "l2": "working set > L2 (3 state arrays + mu, w0, mask = 205 MB vs 126 MB L2); each step is a full cold solve",
                   "certified_last_step": n_cert, "certified_all_timed_steps": certified, "accounts": A,
                   "value_counts": "certified accounts only (status 0: scaled residuals <= 1e-6 and gates pass)",
                   "iters_p50": float(np.median(iters)), "iters_max": int(iters.max()),
                   "iterations_per_sec": iters_total / (interval_ms * 1e-3) if interval_ms else None,
                   "max_scaled_residual": float(max(resid[:, 7].max(), resid[:, 8].max())),
                   "max_gate_residual": float(resid[:, 0:4].max()), "device_bytes": P.device_bytes, "library": pr.version(),
                   "create_plus_first_solve_ms": create_plus_solve_ms,
                   "accounts_per_s_incl_create": A / (create_plus_solve_ms * 1e-3)},
        "clocks": clocks,
        "e2e": {"value": e2e_cert * world / (e2e_ms * 1e-3), "unit": "accounts/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / args.steps,
                "note": "prism_solve_batch_host: mu and w0 go host->device every step; bounds, masks, bands, tau, gamma and the "
                        "universe stay resident from prism_problem_create"},
        "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "extra": extra,
    }
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
