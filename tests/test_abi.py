"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU and exports every
symbol include/prism.h declares; settings defaults; struct layouts of the binding match the header; the product
path has no CPU fallback.  No compute calls (there is no GPU here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_23367_b200 import build, binding
    build.build()
    return binding.load_library()


def _header():
    with open(os.path.join(ROOT, "include", "prism.h")) as f:
        return f.read()


def test_every_declared_symbol_is_exported(lib):
    h = _header()
    names = set(re.findall(r"\b(prism_[a-z0-9_]+)\s*\(", h))
    names -= {"prism_problem", "prism_settings", "prism_data", "prism_constraint_set", "prism_solve_info"}
    assert {"prism_problem_create", "prism_solve_batch", "prism_residuals"} <= names      # BASELINE.json:north_star
    for n in sorted(names):
        assert hasattr(lib, n), f"{n} declared in prism.h but not exported"
    from paper_2606_23367_b200 import binding
    assert set(binding.SYMBOLS) == names


def test_default_settings_and_version(lib):
    from paper_2606_23367_b200 import binding
    s = binding.default_settings()
    assert s.eps_rel == 1e-6 and s.max_iter == 4000 and s.check_every == 10 and s.alpha == 1.6 and s.rho_scale == 100.0
    assert s.adapt_rho == 1 and s.gemm_precision == 3 and s.profile == 0 and s.eps_abs == 0.0 and s.first_check == 40
    assert not s.warm_w and not s.warm_duals
    assert "sm_100a" in binding.version()


def test_header_constants_match_binding():
    from paper_2606_23367_b200 import binding
    from instances import gen
    h = _header()
    assert int(re.search(r"PRISM_NRES = (\d+)", h).group(1)) == binding.NRES
    for name, val in [("PRISM_R_BUDGET", binding.RES["budget"]), ("PRISM_R_STAT", binding.RES["stat"]),
                      ("PRISM_R_OBJECTIVE", binding.RES["objective"]), ("PRISM_R_DUAL", binding.RES["dual"])]:
        assert int(re.search(name + r" = (\d+)", h).group(1)) == val
    flags = dict(re.findall(r"(PRISM_[A-Z_]+) = (\d+)", h))
    assert int(flags["PRISM_GROUP_BANDS"]) == gen.F_GROUP_BANDS and int(flags["PRISM_TAX_LOTS"]) == gen.F_TAX_LOTS
    assert int(flags["PRISM_BENCHMARK_SHIFT"]) == gen.F_BENCHMARK_SHIFT and int(flags["PRISM_EXCLUSION"]) == gen.F_EXCLUSION
    assert len(binding.STATUS_NAMES) == 6                                               # Table 14
    # struct sizes (natural alignment) as the C compiler lays them out
    assert C.sizeof(binding.Settings) == 112 and C.sizeof(binding.ConstraintSet) == 16
    assert C.sizeof(binding.Data) == 22 * 8


def test_struct_sizes_match_the_c_compiler(tmp_path):
    """The ctypes mirrors in binding.py against sizeof() of include/prism.h as gcc lays the structs out."""
    import shutil
    import subprocess
    from paper_2606_23367_b200 import binding
    if shutil.which("gcc") is None:
        pytest.skip("gcc not available")
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include "prism.h"\nint main(void) { printf("%zu %zu %zu %zu\\n", sizeof(prism_settings), '
                   'sizeof(prism_constraint_set), sizeof(prism_data), sizeof(prism_solve_info)); return 0; }\n')
    exe = tmp_path / "sz"
    inc = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include")
    subprocess.run(["gcc", "-I", inc, str(src), "-o", str(exe)], check=True)
    sizes = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert sizes == [C.sizeof(binding.Settings), C.sizeof(binding.ConstraintSet), C.sizeof(binding.Data), C.sizeof(binding.SolveInfo)]


def test_invalid_arguments_are_errors_not_crashes(lib):
    from paper_2606_23367_b200 import binding
    out = C.c_void_p()
    rc = lib.prism_problem_create(10, 2, 1, None, None, None, C.byref(out))
    assert rc == 1 and not out.value and b"null" in lib.prism_last_error()
    cs = binding.ConstraintSet(flags=0, G=0, max_lots=0, prox_form=0)
    d = binding.Data()
    rc = lib.prism_problem_create(10, 2, 1, C.byref(cs), C.byref(d), None, C.byref(out))
    assert rc == 1 and b"mandatory" in lib.prism_last_error()
    cs = binding.ConstraintSet(flags=3, G=0, max_lots=0, prox_form=0)
    rc = lib.prism_problem_create(0, 2, 1, C.byref(cs), C.byref(d), None, C.byref(out))
    assert rc == 1
    rc = lib.prism_problem_create(10, 1000, 1, C.byref(cs), C.byref(d), None, C.byref(out))
    assert rc == 1
    assert lib.prism_solve_batch(None, None, None, None, None, None, None, None, None) == 4    # PRISM_ERR_NOT_READY
    assert lib.prism_residuals(None, None, None, None, None) == 4
    lib.prism_problem_destroy(None)                                                         # NULL is allowed
    assert lib.prism_problem_device_bytes(None) == 0


def test_product_path_does_not_touch_the_oracle_or_any_cpu_fallback():
    pkg = os.path.join(ROOT, "paper_2606_23367_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f"{fn} mentions the oracle"
    from paper_2606_23367_b200 import binding
    with pytest.raises(RuntimeError):
        binding._lib = None
        try:
            binding.load_library("/nonexistent/libprism.so")
        finally:
            binding._lib = None


def test_shard_plan_covers_every_account_once():
    """paper_2606_23367_b200.shard.account_range: contiguous, balanced, disjoint, complete."""
    from paper_2606_23367_b200 import shard
    for A in (0, 1, 2, 5, 32, 100, 500, 501):
        for world in (1, 2, 3, 4, 8):
            blocks = shard.plan(A, world)
            assert blocks[0][0] == 0 and blocks[-1][1] == A
            assert all(blocks[r][1] == blocks[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1 and sum(sizes) == A
    with pytest.raises(ValueError):
        shard.account_range(4, 2, 2)
    from instances import gen
    inst = gen.config2(N=64, k=4, A=5, G=3)
    sub = shard.slice_instance(inst, 1, 4)
    assert sub.A == 3 and sub.mu.shape == (3, 64) and sub.B is inst.B and sub.band_lo.shape == (3, 3)
    assert (sub.w0 == inst.w0[1:4]).all() and (sub.tau == inst.tau[1:4]).all()


def test_sharded_solve_world_size_2_gloo(tmp_path):
    """Multi-GPU path through the PRODUCT code paper_2606_23367_b200.shard on gloo, world size 2:
    every rank takes its block of one batch, a stand-in block solver returns per-account rows computed from the
    block's own data, and the gathered result must equal the same rows computed on the whole batch, in account order.
    The only communication is the gather (and the barrier / max-reduction bench.py uses for its timings)."""
    import subprocess, sys, textwrap
    code = textwrap.dedent("""
        import os, sys, numpy as np, torch, torch.distributed as dist
        sys.path.insert(0, %r)
        from instances import gen
        from paper_2606_23367_b200 import shard
        dist.init_process_group('gloo')
        r, w = dist.get_rank(), dist.get_world_size()
        inst = gen.config1(seed=0, N=64, k=4, A=5)             # one batch, the same on every rank (strong scaling)
        def rows(sub):                                         # stand-in for Problem(sub).solve(): one row per account
            return {'sig': torch.tensor(np.stack([sub.mu.sum(1), sub.w0.max(1), sub.tau], 1)),
                    'n': torch.tensor(np.full((sub.A, 1), sub.A, dtype=np.int64))}
        out = shard.solve_sharded(inst, rows)
        want = rows(inst)['sig']
        assert out['sig'].shape == (5, 3) and torch.equal(out['sig'], want), (out['sig'], want)
        a, b = shard.account_range(inst.A, w, r)
        assert (out['n'][a:b] == b - a).all() and int(out['n'].sum()) == 3 * 3 + 2 * 2
        t = torch.tensor([float(10 + r)], dtype=torch.float64)  # bench.py: barrier + max over ranks of the timing
        dist.barrier()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == 10 + w - 1
        dist.destroy_process_group()
        print('rank' + str(r) + 'done', flush=True)
    """ % ROOT)
    script = tmp_path / "worker.py"
    script.write_text(code)
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29532", str(script)],
                         capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    assert "rank0done" in res.stdout and "rank1done" in res.stdout


def test_queue_layer_identity_and_summary():
    """NEXT-3 host layer (paper_2606_23367_b200.queue_layer): the input identity is deterministic and account-specific, the
    summary reproduces Table 8's columns from the audit records."""
    from instances import gen
    from paper_2606_23367_b200 import queue_layer as ql
    inst = gen.config2(N=64, k=4, A=3, G=3)
    ids = [ql.input_identity(inst, a) for a in range(3)]
    assert len(set(ids)) == 3 and ids == [ql.input_identity(gen.config2(N=64, k=4, A=3, G=3), a) for a in range(3)]
    inst.mu[1, 5] += 1e-9
    assert ql.input_identity(inst, 1) != ids[1] and ql.input_identity(inst, 0) == ids[0]
    recs = [ql.AuditRecord(a, a // 2, "i", "o", st, ql.STATUS_NAMES[st], 10, (0.0,) * 12, lat, 1.0, lat > 25.0, "b")
            for a, (st, lat) in enumerate([(0, 10.0), (0, 10.0), (1, 20.0), (3, 30.0)])]
    s = ql.summarise(recs)
    assert s["accounts"] == 4 and s["completed"] == 4 and s["certified"] == 2 and s["missed_deadline_rate"] == 0.25
    assert s["latency_max_ms"] == 30.0 and abs(s["accounts_per_s"] - 4 / 0.030) < 1e-9 and s["latency_p50_ms"] == 15.0


def test_library_exports_exactly_the_declared_symbols(lib):
    """nm -D: the dynamic symbol table of libprism.so holds the functions include/prism.h declares and nothing else
    (the library is built with hidden default visibility)."""
    import subprocess
    from paper_2606_23367_b200 import binding
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = {l.split()[2] for l in out.splitlines() if len(l.split()) == 3 and l.split()[1] == "T"}
    declared = set(re.findall(r"\b(prism_[a-z0-9_]+)\s*\(", _header()))
    declared -= {"prism_problem", "prism_settings", "prism_data", "prism_constraint_set", "prism_solve_info"}
    assert exported == declared, (sorted(exported - declared), sorted(declared - exported))
