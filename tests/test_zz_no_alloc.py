"""The one entry point that allocates nothing (prism_factor_exposures_noalloc, csrc/k_noalloc.cu): its split-K partials
live in a static __device__ array instead of cudaMalloc'd workspace.  Collected last on purpose (file name): the
suite runs with pytest -x, a failure here must not hide other tests.

Checks: same output as the existing path (prism_factor_exposures: the problem object's GEMM-1 with its create-time
workspace) on two calls in a row with different inputs - the shared scratch keeps the first call's contents, the second
must not see them; no device memory is allocated by the calls; oversize requests are rejected with a clear error."""
import ctypes as C

import numpy as np
import pytest

from instances import gen

pytestmark = pytest.mark.gpu

TOL = 1e-12        # same bar as test_dmma_and_fma_gemms_agree: both sides are fp64, only the summation order differs


def test_noalloc_matches_existing_path_two_calls_in_a_row():
    import torch
    import paper_2606_23367_b200 as pr
    from paper_2606_23367_b200 import binding
    inst = gen.config1(N=3000, k=30, A=40)                      # several split-K chunks, ragged last chunk
    P = pr.Problem(inst)
    dev = P.dev
    B = P.t["B"]
    rng = np.random.default_rng(0)
    X1 = torch.as_tensor(inst.w0).to(dev)                      # first call: the accounts' current weights
    X2 = torch.as_tensor(rng.standard_normal(inst.w0.shape)).to(dev)   # second call: different data, larger magnitudes
    out = torch.full((inst.A, inst.k), float("nan"), dtype=torch.float64, device=dev)
    assert binding.lib().prism_noalloc_init() == 0
    torch.cuda.synchronize()
    for X in (X1, X2):
        ref = P.factor_exposures(X)                             # existing path (allocates nothing either, but owns Tpart)
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated(dev)
        free_before = torch.cuda.mem_get_info(dev)[0]
        binding.factor_exposures_noalloc(B, X, out)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(dev) == before
        assert torch.cuda.mem_get_info(dev)[0] == free_before   # the driver handed out no device memory either
        scale = float(ref.abs().max())
        assert float((out - ref).abs().max()) <= TOL * max(scale, 1.0), float((out - ref).abs().max())
        # and both agree with a plain library matmul
        mm = X @ B.to(torch.float64)
        assert float((out - mm).abs().max()) <= 1e-11 * max(scale, 1.0)
    P.close()


def test_noalloc_fp32_loadings_and_single_chunk():
    import torch
    from paper_2606_23367_b200 import binding
    rng = np.random.default_rng(1)
    B = torch.as_tensor(rng.standard_normal((100, 7)).astype(np.float32)).cuda()       # N < 256: one chunk
    X = torch.as_tensor(rng.standard_normal((3, 100))).cuda()
    out = torch.empty((3, 7), dtype=torch.float64, device="cuda")
    binding.factor_exposures_noalloc(B, X, out)
    torch.cuda.synchronize()
    assert float((out - X @ B.to(torch.float64)).abs().max()) <= 1e-12


def test_noalloc_rejects_sizes_beyond_the_static_scratch():
    import torch
    from paper_2606_23367_b200 import binding
    lib = binding.lib()
    d = torch.zeros(8, dtype=torch.float64, device="cuda")      # never touched: the size check comes first
    A, k = 8192, 128                                            # 1,048,576 > PRISM_NOALLOC_SCRATCH_DOUBLES
    assert A * k > binding.NOALLOC_SCRATCH_DOUBLES
    rc = lib.prism_factor_exposures_noalloc(d.data_ptr(), 0, d.data_ptr(), 10, k, A, None, d.data_ptr())
    assert rc == 1                                              # PRISM_ERR_INVALID_ARG
    msg = lib.prism_last_error().decode()
    assert "PRISM_NOALLOC_SCRATCH_DOUBLES" in msg and "4 MiB" in msg, msg
    assert lib.prism_factor_exposures_noalloc(None, 0, d.data_ptr(), 10, 2, 2, None, d.data_ptr()) == 1
    torch.cuda.synchronize()
