"""Test helper: the CPU oracle on several accounts of one seeded batch at once, one account per worker process
(accounts are independent programs).  Lives under tests/ - only tests may execute oracle/."""
import multiprocessing as mp
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
_INST = {}


_LIMIT = []


def _init(root):
    """One BLAS thread per worker (the parallelism is over accounts): environment first, in case numpy is not loaded
    yet, then threadpoolctl on the libraries that are."""
    for v in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS"):
        os.environ[v] = "1"
    if root not in sys.path:
        sys.path.insert(0, root)
    try:
        import numpy  # noqa: F401  (loads the BLAS that threadpoolctl then limits)
        from threadpoolctl import threadpool_limits
        _LIMIT.append(threadpool_limits(limits=1))
    except Exception:
        pass


def _one(args):
    cfg, seed, kw, a = args
    _init(ROOT)
    from instances import gen
    from oracle import ipm, problem
    key = (cfg, seed, tuple(sorted(kw.items())))
    if key not in _INST:
        _INST.clear()
        _INST[key] = gen.by_name(cfg, seed=seed, **kw)
    inst = _INST[key]
    r = ipm.solve(problem.account_from_instance(inst, a), witness=inst.witness[a])
    return a, r["status"], r["w"], r["mult"]


def solve_accounts(cfg, seed, accounts, procs=None, **kw):
    """Oracle weights, multipliers and statuses of the listed accounts of gen.by_name(cfg, seed, **kw):
    (W, list of dict(mult, status)).  An account on which the oracle reports failure keeps its status: the caller decides."""
    import numpy as np
    procs = procs or max(1, min(os.cpu_count() or 1, len(accounts), 32))
    with mp.get_context("spawn").Pool(procs, initializer=_init, initargs=(ROOT,)) as pool:
        out = pool.map(_one, [(cfg, seed, kw, int(a)) for a in accounts], chunksize=1)
    return np.array([w for _, _, w, _ in out]), [dict(mult=m, status=st) for _, st, _, m in out]
