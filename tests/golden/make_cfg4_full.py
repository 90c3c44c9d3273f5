"""Writes tests/golden/cfg4_full_a{a}.npz: oracle weights of accounts of configs[4] at FULL width (32 x 384,800, seed 0).

Calls only instances/ (seeded generator) and oracle/ (structured interior point, as it stands): no value comes from the
CUDA path.  The oracle needs many minutes per account at this width, which is why the values are stored instead of
being recomputed inside the GPU test (tests/test_gpu_parity.py::test_full_size_cfg4_elementwise).
Stored per account: the full weight vector rounded to float32 (weights <= 1e-3: 6e-11 absolute, against a parity
tolerance of 1e-4; zlib-compressed npz), the oracle's objective, its KKT
certificate (kkt_check with the oracle's multipliers) and the SHA-256 of the account's mu / w0 rows (generator drift).

    python tests/golden/make_cfg4_full.py [account ...]        (default: 0)
"""
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from instances import gen            # noqa: E402
from oracle import ipm, kkt_check, problem   # noqa: E402


def main():
    accounts = [int(x) for x in sys.argv[1:]] or [0]
    inst = gen.by_name("cfg4", seed=0)
    for a in accounts:
        acc = problem.account_from_instance(inst, a)
        t0 = time.perf_counter()
        r = ipm.solve(acc, witness=inst.witness[a])
        dt = time.perf_counter() - t0
        # At this width the structured interior point stalls just above its own acceptance bar (best merit ~2e-9 against
        # 5e-10): the oracle REPORTS FAILURE and the iterate is stored with that status, its merit and
        # the independent checker's certificate, so that the test can say what it compares with.
        w = r["w"]
        feas = kkt_check.feasibility(acc, w)
        out = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"cfg4_full_a{a}.npz")
        k = kkt_check.kkt(acc, w, r["mult"], delta=1e-7)
        np.savez_compressed(out, w=w.astype(np.float32), objective=problem.objective(acc, w), iterations=r["iters"], status=r["status"],
                            r_stat=k["r_stat"], r_comp=k["r_comp"],
                            seconds=dt, feas=np.array([feas[k] for k in sorted(feas)]),
                            sha_mu=hashlib.sha256(np.ascontiguousarray(inst.mu[a]).tobytes()).hexdigest(),
                            sha_w0=hashlib.sha256(np.ascontiguousarray(inst.w0[a]).tobytes()).hexdigest())
        print(f"account {a}: {r['status']}, r_stat {k['r_stat']:.2e}, {dt:.0f} s, objective {problem.objective(acc, w):.12e}, max feasibility residual "
              f"{max(feas.values()):.2e} -> {out}", flush=True)


if __name__ == "__main__":
    main()
