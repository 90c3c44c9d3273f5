"""queue_layer.py - queue / deadline / audit layer over the batch solver: a thin HOST-side layer, no arithmetic
of the method.

The paper frames its headline result as a production queue (Table 8): M accounts inside a time
window, completion count, missed-deadline rate, p50 / p99 latency, throughput Lambda = M / T_queue, and
one audit record per account (PAPER.md:160-166 record fields, PAPER.md:368 audit artifact): identity of the input and
of the output, elapsed time, status, build id.  Here:

* `run_queue(inst, batch_size, deadline_ms, time_limit_ms, lanes)` cuts the accounts of an instance into consecutive batches
  (`shard.slice_instance`), solves each with one `prism_solve_batch` (cold start) - `lanes` of them
  concurrently, one host thread and one CUDA stream per lane - and stamps every account
  with the time at which its result became available to the caller - the end of its batch's call, measured from the
  start of the queue.  `deadline_ms` / `time_limit_ms` are passed through to the solver per batch (statuses LATE /
  TIMEOUT of the Table 14 vocabulary) AND applied to the queue clock (an account whose batch ends after the queue deadline
  is a missed deadline whatever its solver status).
* `AuditRecord`: SHA-256 of the account's inputs (mu, w0, bounds, tau, gamma, ... in a fixed order) and of the returned
  weights, status, iterations, the residual block, elapsed ms, build id (`prism_version`).
* `solve_concurrently(problems)`: resident problem objects solved at once, one stream each (queue depth > 1 batch).
* `summarise(records)`: completion count, missed-deadline rate, p50 / p99 / max latency, Lambda.
"""
from __future__ import annotations

import dataclasses
import hashlib
import time
from dataclasses import dataclass

import numpy as np

from . import binding, shard

STATUS_NAMES = {0: "certified", 1: "feasible", 2: "timeout", 3: "late", 4: "no_feasible", 5: "failure"}


@dataclass
class AuditRecord:
    account: int                 # index in the queue
    batch: int
    input_sha256: str            # identity of the account's problem data
    output_sha256: str           # identity of the returned weights
    status: int
    status_name: str
    iterations: int
    residuals: tuple             # the PRISM_NRES residual block (gates, KKT residuals, objective, ...)
    latency_ms: float            # queue start -> result available (end of the batch's call)
    solve_interval_ms: float     # device interval of the batch (reported solve interval)
    missed_deadline: bool
    build_id: str


def universe_identity(inst) -> str:
    """SHA-256 of the shared universe (B, f, d, group ids), hashed once per queue."""
    h = hashlib.sha256()
    for name in ("B", "f", "d", "group_id"):
        v = getattr(inst, name)
        if v is not None:
            h.update(name.encode()); h.update(np.ascontiguousarray(v).tobytes())
    return h.hexdigest()


def input_identity(inst, a: int, universe: str = None) -> str:
    """SHA-256 over the universe's digest and the account's own data in a fixed field order."""
    h = hashlib.sha256()
    h.update((universe or universe_identity(inst)).encode())
    for name in shard.PER_ACCOUNT:
        if name in ("witness", "tau_drawn"):
            continue
        v = getattr(inst, name)
        if v is not None:
            h.update(name.encode()); h.update(np.ascontiguousarray(v[a]).tobytes())
    return h.hexdigest()


def run_queue(inst, batch_size: int, deadline_ms: float = 0.0, time_limit_ms: float = 0.0, device: str = "cuda:0",
              lanes: int = 1, **settings):
    """Solves the accounts of `inst` as a queue of consecutive batches; returns (weights (A, N) numpy, list of AuditRecord).

    lanes > 1: that many worker threads, each with its own CUDA stream, take batches from the queue in order and run
    them concurrently (create, solve, read back).  A solve is a chain of short launches whose length is set by the
    slowest account of every launch, so one batch leaves most of the GPU idle; independent batches fill it
    (accounts are independent programs, PAPER.md:124 - there is no exchange between lanes)."""
    import threading
    import torch
    if batch_size < 1 or lanes < 1:
        raise ValueError("batch_size and lanes must be >= 1")
    build = binding.version()
    uni = universe_identity(inst)
    ids = [input_identity(inst, a, uni) for a in range(inst.A)]       # (identity of the inputs: before the clock starts)
    W = np.empty((inst.A, inst.N))
    batches = list(enumerate(range(0, inst.A, batch_size)))
    done, errors, lock, cursor = {}, [], threading.Lock(), [0]
    t0 = time.perf_counter()

    def lane(stream):
        while True:
            with lock:
                i = cursor[0]; cursor[0] += 1
            if i >= len(batches) or errors:
                return
            b, start = batches[i]
            stop = min(inst.A, start + batch_size)
            sub = shard.slice_instance(inst, start, stop)
            P = binding.Problem(sub, device=device)
            left = max(deadline_ms - 1e3 * (time.perf_counter() - t0), 1e-3) if deadline_ms > 0 else 0.0
            r = P.solve(binding.default_settings(deadline_ms=left, time_limit_ms=time_limit_ms, **settings))
            if stream is None:
                torch.cuda.synchronize()
            else:
                stream.synchronize()
            w = r.w.cpu().numpy(); st = r.status.cpu().numpy(); it = r.iters.cpu().numpy(); rs = r.resid.cpu().numpy()
            latency = 1e3 * (time.perf_counter() - t0)
            P.close()
            W[start:stop] = w
            done[b] = (start, stop, w, st, it, rs, latency, float(r.info["solve_interval_ms"]))

    def worker():
        try:
            stream = torch.cuda.Stream(device=device)
            with torch.cuda.stream(stream):
                lane(stream)
        except Exception as e:                                         # re-raised by the caller's thread below
            errors.append(e)

    if lanes == 1:
        lane(None)
    else:
        threads = [threading.Thread(target=worker) for _ in range(min(lanes, len(batches)))]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        if errors:
            raise errors[0]
    records = []
    for b, _ in batches:
        start, stop, w, st, it, rs, latency, interval = done[b]
        for j in range(stop - start):
            a = start + j
            missed = deadline_ms > 0 and (latency > deadline_ms or int(st[j]) in (2, 3))
            records.append(AuditRecord(a, b, ids[a], hashlib.sha256(np.ascontiguousarray(w[j]).tobytes()).hexdigest(),
                                       int(st[j]), STATUS_NAMES.get(int(st[j]), "?"), int(it[j]), tuple(float(x) for x in rs[j]),
                                       latency, interval, bool(missed), build))
    return W, records


def solve_concurrently(problems, **settings):
    """One `prism_solve_batch` per problem object, all at once: one host thread and one CUDA stream per problem.
    Returns (list of SolveResult, wall-clock ms from the first launch to the last result, device idle on both sides).
    For queues deeper than one batch whose problem objects are already resident (the repeated-run lane)."""
    import threading
    import torch
    results, errors = [None] * len(problems), []

    def worker(i):
        try:
            stream = torch.cuda.Stream(device=problems[i].dev)
            with torch.cuda.stream(stream):
                results[i] = problems[i].solve(binding.default_settings(**settings))
                stream.synchronize()
        except Exception as e:
            errors.append(e)

    torch.cuda.synchronize()
    t0 = time.perf_counter()
    threads = [threading.Thread(target=worker, args=(i,)) for i in range(len(problems))]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize()
    ms = 1e3 * (time.perf_counter() - t0)
    if errors:
        raise errors[0]
    return results, ms


def summarise(records) -> dict:
    """Table 8's columns: completion count, missed-deadline rate, latency quantiles, Lambda = M / T_queue."""
    lat = np.array([r.latency_ms for r in records]) if records else np.zeros(1)
    done = sum(1 for r in records if r.status in (0, 1, 3))
    return {"accounts": len(records), "completed": done, "certified": sum(1 for r in records if r.status == 0),
            "missed_deadline_rate": (sum(1 for r in records if r.missed_deadline) / len(records)) if records else 0.0,
            "latency_p50_ms": float(np.percentile(lat, 50)), "latency_p99_ms": float(np.percentile(lat, 99)),
            "latency_max_ms": float(lat.max()), "queue_ms": float(lat.max()),
            "accounts_per_s": len(records) / (lat.max() * 1e-3) if records and lat.max() > 0 else 0.0,
            "build_id": records[0].build_id if records else binding.version()}


def records_as_rows(records) -> list:
    return [dataclasses.asdict(r) for r in records]
