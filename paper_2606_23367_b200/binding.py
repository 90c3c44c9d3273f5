"""ctypes binding of include/prism.h - argument marshalling only; every step of the path runs in the CUDA kernels.

PyTorch supplies device memory (torch.Tensor.data_ptr) and the stream handle; nothing here computes.
The library must exist (build it with `python -m paper_2606_23367_b200.build` or `__graft_entry__.build()`):
there is no CPU fallback, a missing library raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libprism.so")

NRES = 12
RES = dict(budget=0, box=1, exposure=2, turnover=3, stat=4, comp=5, objective=6, primal=7, dual=8,
           turnover_value=9, rho=10)
STATUS_NAMES = ["certified", "feasible/non-certified", "timeout", "deadline exceeded", "no accepted feasible return",
                "allocation/numerical failure"]
SYMBOLS = ["prism_default_settings", "prism_problem_create", "prism_solve_batch", "prism_residuals",
           "prism_solve_batch_host", "prism_problem_destroy", "prism_problem_device_bytes", "prism_last_error",
           "prism_version", "prism_kernel_times", "prism_factor_exposures", "prism_noalloc_init",
           "prism_factor_exposures_noalloc", "prism_fp64_yardstick", "prism_problem_prox_form", "prism_project"]
NOALLOC_SCRATCH_DOUBLES = 524288      # prism.h: PRISM_NOALLOC_SCRATCH_DOUBLES


PROX_AUTO, PROX_RESIDENT, PROX_STREAMING, PROX_EVERY_ASSET = 0, 1, 2, 3     # prism.h: PRISM_PROX_*
GEMM_FP64_TENSOR, GEMM_FP64_FMA = 0, 1                                       # prism.h: PRISM_GEMM_*


class ConstraintSet(C.Structure):
    _fields_ = [("flags", C.c_uint32), ("G", C.c_int32), ("max_lots", C.c_int32), ("prox_form", C.c_int32)]


class Data(C.Structure):
    _fields_ = [("B", C.c_void_p), ("B_is_fp32", C.c_int32), ("f", C.c_void_p), ("d", C.c_void_p),
                ("group_id", C.c_void_p), ("d_t", C.c_void_p), ("mu", C.c_void_p), ("gamma", C.c_void_p),
                ("w0", C.c_void_p), ("w_b", C.c_void_p), ("lo", C.c_void_p), ("hi", C.c_void_p),
                ("hi_full", C.c_void_p), ("excl", C.c_void_p), ("tau", C.c_void_p), ("kappa", C.c_void_p),
                ("band_lo", C.c_void_p), ("band_hi", C.c_void_p), ("c_buy", C.c_void_p), ("lot_slope", C.c_void_p),
                ("lot_width", C.c_void_p), ("lot_count", C.c_void_p)]


class Settings(C.Structure):
    _fields_ = [("eps_rel", C.c_double), ("eps_abs", C.c_double), ("max_iter", C.c_int32), ("check_every", C.c_int32),
                ("first_check", C.c_int32), ("adapt_rho", C.c_int32), ("adapt_start", C.c_int32), ("adapt_every", C.c_int32),
                ("alpha", C.c_double), ("rho_scale", C.c_double),
                ("gemm_precision", C.c_int32), ("profile", C.c_int32), ("time_limit_ms", C.c_double),
                ("deadline_ms", C.c_double), ("prox_window_mult", C.c_double), ("sample_until", C.c_int32),
                ("reserved0", C.c_int32), ("warm_w", C.c_void_p),
                ("warm_duals", C.c_void_p)]


class SolveInfo(C.Structure):
    _fields_ = [("solve_interval_ms", C.c_double), ("wall_ms", C.c_double), ("device_bytes", C.c_int64),
                ("iters_max", C.c_int32), ("iters_total", C.c_int64), ("n_certified", C.c_int32),
                ("n_feasible", C.c_int32), ("n_timeout", C.c_int32), ("n_late", C.c_int32),
                ("n_no_feasible", C.c_int32), ("n_failed", C.c_int32), ("kernel_launches", C.c_int64)]


_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen libprism.so and declare the prototypes.  Raises if the library is missing (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise RuntimeError(f"{path} not found: build the CUDA library first (python -m paper_2606_23367_b200.build); "
                           "there is no CPU fallback")
    L = C.CDLL(path)
    L.prism_default_settings.argtypes = [C.POINTER(Settings)]; L.prism_default_settings.restype = None
    L.prism_problem_create.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.POINTER(ConstraintSet), C.POINTER(Data),
                                       C.c_void_p, C.POINTER(C.c_void_p)]
    L.prism_problem_create.restype = C.c_int
    L.prism_solve_batch.argtypes = [C.c_void_p, C.POINTER(Settings), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.POINTER(SolveInfo)]
    L.prism_solve_batch.restype = C.c_int
    L.prism_residuals.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.prism_residuals.restype = C.c_int
    L.prism_solve_batch_host.argtypes = [C.c_void_p, C.POINTER(Settings), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(SolveInfo)]
    L.prism_solve_batch_host.restype = C.c_int
    L.prism_problem_destroy.argtypes = [C.c_void_p]; L.prism_problem_destroy.restype = None
    L.prism_problem_device_bytes.argtypes = [C.c_void_p]; L.prism_problem_device_bytes.restype = C.c_int64
    L.prism_last_error.argtypes = []; L.prism_last_error.restype = C.c_char_p
    L.prism_version.argtypes = []; L.prism_version.restype = C.c_char_p
    L.prism_kernel_times.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]; L.prism_kernel_times.restype = C.c_int
    L.prism_factor_exposures.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]; L.prism_factor_exposures.restype = C.c_int
    L.prism_project.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]; L.prism_project.restype = C.c_int
    L.prism_noalloc_init.argtypes = []; L.prism_noalloc_init.restype = C.c_int
    L.prism_problem_prox_form.argtypes = [C.c_void_p]; L.prism_problem_prox_form.restype = C.c_int32
    L.prism_fp64_yardstick.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]; L.prism_fp64_yardstick.restype = C.c_int
    L.prism_factor_exposures_noalloc.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_int32, C.c_int32,
                                                 C.c_void_p, C.c_void_p]
    L.prism_factor_exposures_noalloc.restype = C.c_int
    _lib = L
    return L


def lib():
    return load_library()


def version() -> str:
    return lib().prism_version().decode()


def default_settings(**kw) -> Settings:
    s = Settings()
    lib().prism_default_settings(C.byref(s))
    for k, v in kw.items():
        if not hasattr(s, k):
            raise AttributeError(k)
        setattr(s, k, v)
    return s


def _check(rc: int):
    if rc != 0:
        raise RuntimeError(f"prism error {rc}: {lib().prism_last_error().decode()}")


@dataclass
class SolveResult:
    w: "object"          # torch (A, N) float64, device
    status: "object"     # torch (A,) int32
    iters: "object"      # torch (A,) int32
    resid: "object"      # torch (A, NRES) float64
    duals: "object"      # torch (A, 2 + 2G) float64
    info: dict


class Problem:
    """prism_problem_create / prism_solve_batch / prism_residuals on torch CUDA tensors."""

    def __init__(self, inst, device="cuda:0", prox_form=PROX_AUTO):
        import torch
        self.torch = torch
        self.dev = torch.device(device)
        self.inst = inst
        self.N, self.k, self.A, self.G = inst.N, inst.k, inst.A, inst.G
        t = {}

        def up(name, arr, dtype=None):
            if arr is None:
                return None
            x = torch.as_tensor(arr)
            if dtype is not None:
                x = x.to(dtype)
            x = x.contiguous().to(self.dev)
            t[name] = x
            return x
        f64 = torch.float64
        if inst.b_fp32:
            up("B", inst.B, torch.float32)
        else:
            up("B", inst.B, f64)
        up("f", inst.f, f64); up("d", inst.d, f64); up("group_id", inst.group_id, torch.uint8)
        up("mu", inst.mu, f64); up("gamma", inst.gamma, f64); up("w0", inst.w0, f64); up("w_b", inst.w_b, f64)
        up("lo", inst.lo, f64); up("hi", inst.hi, f64); up("hi_full", inst.hi_full, f64); up("excl", inst.excl, torch.uint8)
        up("tau", inst.tau, f64); up("kappa", inst.kappa, f64); up("band_lo", inst.band_lo, f64); up("band_hi", inst.band_hi, f64)
        up("c_buy", inst.c_buy, f64); up("lot_slope", inst.lot_slope, f64); up("lot_width", inst.lot_width, f64)
        up("lot_count", inst.lot_count, torch.uint8)
        self.t = t
        d = Data()
        for name, _ in Data._fields_:
            if name == "B_is_fp32":
                d.B_is_fp32 = 1 if inst.b_fp32 else 0
            elif name == "d_t":
                d.d_t = None
            else:
                x = t.get(name)
                setattr(d, name, x.data_ptr() if x is not None else None)
        self.cs = ConstraintSet(flags=int(inst.flags), G=int(inst.G), max_lots=4 if inst.lot_slope is not None else 0,
                                prox_form=int(prox_form))
        self.handle = C.c_void_p()
        with torch.cuda.device(self.dev):
            stream = torch.cuda.current_stream().cuda_stream
            _check(lib().prism_problem_create(self.N, self.k, self.A, C.byref(self.cs), C.byref(d), C.c_void_p(stream),
                                              C.byref(self.handle)))
        self.data = d

    def close(self):
        if getattr(self, "handle", None) is not None and self.handle.value:
            lib().prism_problem_destroy(self.handle)
            self.handle = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def prox_form(self) -> int:
        return int(lib().prism_problem_prox_form(self.handle))

    @property
    def device_bytes(self) -> int:
        return int(lib().prism_problem_device_bytes(self.handle))

    def _info(self, info: SolveInfo) -> dict:
        return {n: getattr(info, n) for n, _ in SolveInfo._fields_}

    def solve(self, settings: Optional[Settings] = None, warm=None, **kw) -> SolveResult:
        """prism_solve_batch.  warm: a previous SolveResult (or (w, duals) device tensors) to warm-start from."""
        torch = self.torch
        s = settings if settings is not None else default_settings(**kw)
        if warm is not None:
            ww, wd = (warm.w, warm.duals) if isinstance(warm, SolveResult) else warm
            self._warm = (ww.contiguous(), None if wd is None else wd.contiguous())       # keep alive during the call
            s.warm_w = self._warm[0].data_ptr()
            s.warm_duals = self._warm[1].data_ptr() if self._warm[1] is not None else None
        w = torch.empty((self.A, self.N), dtype=torch.float64, device=self.dev)
        status = torch.empty(self.A, dtype=torch.int32, device=self.dev)
        iters = torch.empty(self.A, dtype=torch.int32, device=self.dev)
        resid = torch.empty((self.A, NRES), dtype=torch.float64, device=self.dev)
        duals = torch.empty((self.A, 2 + 2 * self.G), dtype=torch.float64, device=self.dev)
        info = SolveInfo()
        with torch.cuda.device(self.dev):
            stream = torch.cuda.current_stream().cuda_stream
            _check(lib().prism_solve_batch(self.handle, C.byref(s), C.c_void_p(stream), w.data_ptr(), status.data_ptr(),
                                           iters.data_ptr(), resid.data_ptr(), duals.data_ptr(), C.byref(info)))
        return SolveResult(w, status, iters, resid, duals, self._info(info))

    KERNELS = ["prox", "gemm1", "solve", "gemm2", "factor", "diag", "other", "prox_root"]

    def kernel_times(self) -> dict:
        ms = (C.c_double * 8)(); cnt = (C.c_int64 * 8)()
        _check(lib().prism_kernel_times(self.handle, ms, cnt))
        return {n: dict(ms=ms[i], launches=int(cnt[i])) for i, n in enumerate(self.KERNELS)}

    def fp64_yardstick(self) -> dict:
        """prism_fp64_yardstick: measured fp64 TFLOP/s of this device (tensor pipe DMMA, FMA pipe)."""
        out = (C.c_double * 2)()
        with self.torch.cuda.device(self.dev):
            stream = self.torch.cuda.current_stream().cuda_stream
            _check(lib().prism_fp64_yardstick(self.handle, C.c_void_p(stream), out))
        return dict(dmma_tflops=out[0], fma_tflops=out[1])

    def factor_exposures(self, w):
        """prism_factor_exposures: (A, k) = w B through the problem's own GEMM-1."""
        torch = self.torch
        w = torch.as_tensor(w, dtype=torch.float64).contiguous().to(self.dev)
        out = torch.empty((self.A, self.k), dtype=torch.float64, device=self.dev)
        with torch.cuda.device(self.dev):
            stream = torch.cuda.current_stream().cuda_stream
            _check(lib().prism_factor_exposures(self.handle, w.data_ptr(), C.c_void_p(stream), out.data_ptr()))
        return out

    def project(self, v, rho_scale: float = 100.0):
        """prism_project: one exact application of the fused projection to the points v (A, N); returns (z, duals)."""
        torch = self.torch
        v = torch.as_tensor(v, dtype=torch.float64).contiguous().to(self.dev)
        z = torch.empty((self.A, self.N), dtype=torch.float64, device=self.dev)
        duals = torch.empty((self.A, 2 + 2 * self.G), dtype=torch.float64, device=self.dev)
        with torch.cuda.device(self.dev):
            stream = torch.cuda.current_stream().cuda_stream
            _check(lib().prism_project(self.handle, v.data_ptr(), C.c_double(rho_scale), C.c_void_p(stream), z.data_ptr(),
                                       duals.data_ptr()))
        return z, duals

    def residuals(self, w, duals=None):
        torch = self.torch
        w = torch.as_tensor(w, dtype=torch.float64).contiguous().to(self.dev)
        if duals is not None:
            duals = torch.as_tensor(duals, dtype=torch.float64).contiguous().to(self.dev)
        resid = torch.empty((self.A, NRES), dtype=torch.float64, device=self.dev)
        with torch.cuda.device(self.dev):
            stream = torch.cuda.current_stream().cuda_stream
            _check(lib().prism_residuals(self.handle, w.data_ptr(), duals.data_ptr() if duals is not None else None,
                                         C.c_void_p(stream), resid.data_ptr()))
        return resid

    def solve_host(self, mu_host, w0_host, w_host, status_host, iters_host, resid_host, settings: Optional[Settings] = None):
        """End-to-end lane: host (pinned) buffers in and out, copies inside the call (prism_solve_batch_host)."""
        torch = self.torch
        s = settings if settings is not None else default_settings()
        info = SolveInfo()

        def ptr(x):
            return x.data_ptr() if x is not None else None
        with torch.cuda.device(self.dev):
            stream = torch.cuda.current_stream().cuda_stream
            _check(lib().prism_solve_batch_host(self.handle, C.byref(s), C.c_void_p(stream), ptr(mu_host), ptr(w0_host),
                                                ptr(w_host), ptr(status_host), ptr(iters_host), ptr(resid_host),
                                                C.byref(info)))
        return self._info(info)


def factor_exposures_noalloc(B, X, out):
    """prism_factor_exposures_noalloc on caller-owned CUDA tensors (B: (N, k) fp64 or fp32, X: (A, N) fp64, out: (A, k)
    fp64, all contiguous).  Allocates nothing; asynchronous on the current stream."""
    import torch
    N, k = B.shape
    A = X.shape[0]
    assert X.shape[1] == N and tuple(out.shape) == (A, k) and B.is_contiguous() and X.is_contiguous() and out.is_contiguous()
    assert X.dtype == torch.float64 and out.dtype == torch.float64 and B.dtype in (torch.float64, torch.float32)
    with torch.cuda.device(X.device):
        stream = torch.cuda.current_stream().cuda_stream
        _check(lib().prism_factor_exposures_noalloc(B.data_ptr(), 1 if B.dtype == torch.float32 else 0, X.data_ptr(), N, k, A,
                                                    C.c_void_p(stream), out.data_ptr()))
    return out
