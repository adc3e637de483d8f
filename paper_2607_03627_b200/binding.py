"""ctypes binding of include/uc_pdhg.h (same names, argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

OPTIMAL, ITERATION_LIMIT, CANCELLED, TIME_LIMIT, NUMERICAL_ERROR = 0, 1, 2, 3, 4
STATUS_NAMES = {0: "OPTIMAL", 1: "ITERATION_LIMIT", 2: "CANCELLED", 3: "TIME_LIMIT", 4: "NUMERICAL_ERROR"}


class UcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"uc_pdhg error {code}: {msg}")
        self.code = code


class Options(C.Structure):
    _fields_ = [("device", C.c_int32), ("ruiz_iters", C.c_int32), ("pc_alpha", C.c_double),
                ("sell_window", C.c_int32), ("long_row_threshold", C.c_int32),
                ("keep_source_map", C.c_int32), ("index_compression", C.c_int32), ("host_ingest", C.c_int32), ("max_ctas", C.c_int32)]


class Params(C.Structure):
    _fields_ = [("iter_limit", C.c_int64), ("eps_rel", C.c_double), ("eps_abs", C.c_double),
                ("time_limit_s", C.c_double), ("check_every", C.c_int32), ("pad_", C.c_int32),
                ("fixed_iterations", C.c_int64), ("beta_sufficient", C.c_double), ("beta_necessary", C.c_double),
                ("beta_artificial", C.c_double), ("weight_smoothing", C.c_double),
                ("x0", C.c_void_p), ("y0", C.c_void_p), ("stream", C.c_void_p),
                ("attempt_trace", C.c_void_p), ("attempt_trace_cap", C.c_int64),
                ("check_trace", C.c_void_p), ("check_trace_cap", C.c_int64),
                ("eta0", C.c_double), ("omega0", C.c_double)]


class Result(C.Structure):
    _fields_ = [("status", C.c_int32), ("returned_average", C.c_int32), ("iterations", C.c_int64),
                ("accepted", C.c_int64), ("restarts", C.c_int64), ("rel_kkt", C.c_double),
                ("rel_primal_res", C.c_double), ("rel_dual_res", C.c_double), ("rel_gap", C.c_double),
                ("primal_obj", C.c_double), ("dual_obj", C.c_double), ("eta", C.c_double), ("omega", C.c_double),
                ("solve_seconds", C.c_double), ("loop_seconds", C.c_double),
                ("attempt_records", C.c_int64), ("check_records", C.c_int64), ("kernel_launches", C.c_int64)]


class Info(C.Structure):
    _fields_ = [("m", C.c_int64), ("n", C.c_int64), ("nnz", C.c_int64),
                ("k_sell_slots", C.c_int64), ("kt_sell_slots", C.c_int64),
                ("k_long_rows", C.c_int64), ("kt_long_rows", C.c_int64),
                ("k_long_nnz", C.c_int64), ("kt_long_nnz", C.c_int64), ("device_bytes", C.c_int64),
                ("precondition_seconds", C.c_double), ("create_seconds", C.c_double),
                ("eta0", C.c_double), ("omega0", C.c_double), ("norm_b", C.c_double), ("norm_c", C.c_double),
                ("bytes_per_attempt", C.c_int64), ("k_narrow_slots", C.c_int64), ("kt_narrow_slots", C.c_int64),
                ("scratch_cached_bytes", C.c_int64)]


ATTEMPT_DTYPE = np.dtype([("eta_used", "f8"), ("eta_bar", "f8"), ("eta_next", "f8"), ("dx2", "f8"),
                          ("dy2", "f8"), ("inter", "f8"), ("accepted", "i4"), ("pad_", "i4")])
CHECK_DTYPE = np.dtype([("k", "i8"), ("restart_kind", "i4"), ("candidate", "i4"), ("omega_after", "f8"),
                        ("mu_c", "f8"), ("mu_r", "f8"), ("relkkt_cur", "f8"), ("relkkt_avg", "f8")])

SPMV_STATIC_MAX_DOUBLES = 262144      # UC_SPMV_STATIC_MAX_DOUBLES of include/uc_pdhg.h

EXPORTS = ["uc_lp_default_options", "uc_lp_create", "uc_lp_update_bounds", "uc_lp_update_objective", "uc_lp_destroy", "uc_release_scratch",
           "uc_pdhg_default_params", "uc_pdhg_solve", "uc_pdhg_solve_device", "uc_pdhg_solve_batch", "uc_pdhg_cancel", "uc_pdhg_cancel_clear", "uc_pdhg_time_kernels", "uc_pdhg_timeline", "uc_lp_compare_layout",
           "uc_lp_get_info", "uc_lp_get_scaling", "uc_lp_get_scaled_values", "uc_lp_spmv", "uc_lp_spmv_static", "uc_last_error",
           "uc_host_log_rounded", "uc_host_exp_rounded", "uc_host_layout_selftest"]

_lib = None


def library_path() -> str:
    return _build.LIB


def load_library(build_if_missing: bool = True):
    """dlopen the compiled extension; fails loudly when it is absent (there is no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path):
        if not build_if_missing:
            raise UcError(-2, f"{path} is missing: run __graft_entry__.build() (no CPU fallback exists)")
        _build.build()
    lib = C.CDLL(path)
    for name in EXPORTS:
        getattr(lib, name)                      # AttributeError if a declared symbol is not exported
    lib.uc_last_error.restype = C.c_char_p
    for f in (lib.uc_host_log_rounded, lib.uc_host_exp_rounded):
        f.restype = C.c_double
        f.argtypes = [C.c_double]
    lib.uc_lp_destroy.restype = None
    lib.uc_lp_destroy.argtypes = [C.c_void_p]
    lib.uc_pdhg_cancel.argtypes = [C.c_void_p]
    lib.uc_lp_create.argtypes = [C.c_int64, C.c_int64, C.c_int64] + [C.c_void_p] * 10
    lib.uc_lp_update_bounds.argtypes = [C.c_void_p] * 3
    lib.uc_lp_update_objective.argtypes = [C.c_void_p] * 2
    lib.uc_pdhg_solve.argtypes = [C.c_void_p] * 5
    lib.uc_pdhg_solve_device.argtypes = [C.c_void_p] * 5
    lib.uc_pdhg_solve_batch.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32]
    lib.uc_pdhg_time_kernels.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.uc_pdhg_timeline.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.uc_host_layout_selftest.argtypes = [C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_int32, C.c_int32, C.c_int32, C.c_int32]
    lib.uc_lp_get_info.argtypes = [C.c_void_p] * 2
    lib.uc_lp_get_scaling.argtypes = [C.c_void_p] * 3
    lib.uc_lp_get_scaled_values.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    lib.uc_lp_spmv.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.uc_pdhg_cancel_clear.argtypes = [C.c_void_p, C.c_void_p]
    lib.uc_release_scratch.argtypes = [C.c_int32, C.c_void_p]
    lib.uc_lp_spmv_static.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    _lib = lib
    return lib


def _check(rc):
    if rc != 0:
        raise UcError(rc, load_library().uc_last_error().decode())


def host_layout_selftest(lp, sell_window=4096, long_row_threshold=32, sched_ctas=148, warps_per_cta=15) -> None:
    """uc_host_layout_selftest on a workloads.LP; raises UcError with the violated property."""
    lib = load_library()
    rp = np.ascontiguousarray(lp.row_ptr, dtype=np.int64); ci = np.ascontiguousarray(lp.col_idx, dtype=np.int32)
    va = np.ascontiguousarray(lp.val, dtype=np.float64)
    _check(lib.uc_host_layout_selftest(int(lp.m), int(lp.n), int(lp.nnz), C.c_void_p(rp.ctypes.data), C.c_void_p(ci.ctypes.data),
                                       C.c_void_p(va.ctypes.data), int(sell_window), int(long_row_threshold), int(sched_ctas), int(warps_per_cta)))


def release_scratch(device: int = -1) -> int:
    """uc_release_scratch: free the per-device scratch block that uc_lp_create keeps cached; returns the bytes freed."""
    n = C.c_int64(0)
    _check(load_library().uc_release_scratch(int(device), C.cast(C.byref(n), C.c_void_p)))
    return int(n.value)


def default_options(**kw) -> Options:
    o = Options()
    load_library().uc_lp_default_options(C.byref(o))
    for k, v in kw.items():
        assert hasattr(o, k), k
        setattr(o, k, v)
    return o


def default_params(**kw) -> Params:
    p = Params()
    load_library().uc_pdhg_default_params(C.byref(p))
    for k, v in kw.items():
        assert hasattr(p, k), k
        setattr(p, k, v)
    return p


def _host(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, C.c_void_p(a.ctypes.data if a.size else None)


@dataclass
class Solution:
    x: object
    y: object
    status: int
    returned_average: int
    iterations: int
    accepted: int
    restarts: int
    rel_kkt: float
    rel_primal_res: float
    rel_dual_res: float
    rel_gap: float
    primal_obj: float
    dual_obj: float
    eta: float
    omega: float
    solve_seconds: float
    loop_seconds: float
    kernel_launches: int
    attempts: np.ndarray
    checks: np.ndarray


def solve_batch(handles, max_concurrent=0, want_xy=True, **params):
    """uc_pdhg_solve_batch: solve the LPs of `handles` (UcLp objects) concurrently; returns one Solution per handle."""
    lib = load_library()
    k = len(handles)
    prm = default_params(**params)
    hs = (C.c_void_p * k)(*[h._h for h in handles])
    xs = [np.zeros(h.n) if want_xy else None for h in handles]
    ys = [np.zeros(h.m) if want_xy else None for h in handles]
    px = (C.c_void_p * k)(*[C.c_void_p(x.ctypes.data) if want_xy and x.size else None for x in xs]) if want_xy else None
    py = (C.c_void_p * k)(*[C.c_void_p(y.ctypes.data) if want_xy and y.size else None for y in ys]) if want_xy else None
    res = (Result * k)()
    _check(lib.uc_pdhg_solve_batch(C.cast(hs, C.c_void_p), k, C.cast(C.byref(prm), C.c_void_p),
                                   C.cast(px, C.c_void_p) if want_xy else None, C.cast(py, C.c_void_p) if want_xy else None,
                                   C.cast(res, C.c_void_p), int(max_concurrent)))
    empty_a, empty_c = np.zeros(0, dtype=ATTEMPT_DTYPE), np.zeros(0, dtype=CHECK_DTYPE)
    return [UcLp._solution(res[i], xs[i], ys[i], empty_a, empty_c, 0, 0) for i in range(k)]


class UcLp:
    """Owner of one uc_lp handle.  `lp` is any object with m, n, row_ptr, col_idx, val, sense, b, c, l, u."""

    def __init__(self, lp, **options):
        self._h = C.c_void_p()
        self.lib = load_library()
        self.m, self.n = int(lp.m), int(lp.n)
        nnz = int(lp.row_ptr[-1]) if len(lp.row_ptr) else 0
        self.nnz = nnz
        keep = []
        args = []
        for arr, dt in ((lp.row_ptr, np.int64), (lp.col_idx, np.int32), (lp.val, np.float64), (lp.sense, np.uint8),
                        (lp.b, np.float64), (lp.c, np.float64), (lp.l, np.float64), (lp.u, np.float64)):
            a, p = _host(arr, dt)
            keep.append(a); args.append(p)
        opt = default_options(**options)
        _check(self.lib.uc_lp_create(self.m, self.n, nnz, *args, C.cast(C.byref(opt), C.c_void_p), C.cast(C.byref(self._h), C.c_void_p)))

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self.lib.uc_lp_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- calls of the ABI, same names
    def uc_pdhg_cancel(self):
        _check(self.lib.uc_pdhg_cancel(self._h))

    cancel = uc_pdhg_cancel

    def uc_pdhg_cancel_clear(self) -> bool:
        """Drop a cancel request kept for the next solve; True if there was one."""
        had = C.c_int32(0)
        _check(self.lib.uc_pdhg_cancel_clear(self._h, C.cast(C.byref(had), C.c_void_p)))
        return bool(had.value)

    cancel_clear = uc_pdhg_cancel_clear

    def uc_lp_update_bounds(self, l, u):
        la, lp_ = _host(l, np.float64)
        ua, up_ = _host(u, np.float64)
        assert la.shape == ua.shape == (self.n,)
        _check(self.lib.uc_lp_update_bounds(self._h, lp_, up_))

    update_bounds = uc_lp_update_bounds

    def uc_lp_update_objective(self, c):
        ca, cp = _host(c, np.float64)
        assert ca.shape == (self.n,)
        _check(self.lib.uc_lp_update_objective(self._h, cp))

    update_objective = uc_lp_update_objective

    def uc_lp_compare_layout(self, lp):
        """Raises UcError unless the device holds, bit for bit, the layouts the host builders make of `lp` (the LP it was created from)."""
        rp = np.ascontiguousarray(lp.row_ptr, dtype=np.int64); ci = np.ascontiguousarray(lp.col_idx, dtype=np.int32)
        va = np.ascontiguousarray(lp.val, dtype=np.float64)
        _check(self.lib.uc_lp_compare_layout(self._h, C.c_int64(self.m), C.c_int64(self.n), C.c_int64(self.nnz), C.c_void_p(rp.ctypes.data),
                                             C.c_void_p(ci.ctypes.data), C.c_void_p(va.ctypes.data)))

    compare_layout = uc_lp_compare_layout

    def uc_pdhg_time_kernels(self, attempts=64, stream=None):
        """(primal_ms, dual_ms): average device time of the two kernels of an attempt (CUDA events)."""
        a, b = C.c_double(0.0), C.c_double(0.0)
        _check(self.lib.uc_pdhg_time_kernels(self._h, C.c_void_p(int(stream)) if stream else None, int(attempts),
                                             C.cast(C.byref(a), C.c_void_p), C.cast(C.byref(b), C.c_void_p)))
        return a.value, b.value

    time_kernels = uc_pdhg_time_kernels

    def uc_pdhg_timeline(self, attempts=16, stream=None):
        """(primal, dual) arrays [grid, 32 warps, 8 marks] of %globaltimer ns for the last of `attempts` attempts
        (a -DUC_TIMELINE build only)."""
        cap = 2 * 1024 * 256
        out = np.zeros(cap, dtype=np.uint64)
        gp, gd = C.c_int32(0), C.c_int32(0)
        _check(self.lib.uc_pdhg_timeline(self._h, C.c_void_p(int(stream)) if stream else None, int(attempts),
                                         out.ctypes.data_as(C.c_void_p), C.c_int64(cap), C.byref(gp), C.byref(gd)))
        a = out[: gp.value * 256].reshape(gp.value, 32, 8)
        b = out[gp.value * 256: (gp.value + gd.value) * 256].reshape(gd.value, 32, 8)
        return a, b

    timeline = uc_pdhg_timeline

    def info(self) -> Info:
        i = Info()
        _check(self.lib.uc_lp_get_info(self._h, C.cast(C.byref(i), C.c_void_p)))
        return i

    def scaling(self):
        Dr = np.zeros(self.m); Dc = np.zeros(self.n)
        _check(self.lib.uc_lp_get_scaling(self._h, C.c_void_p(Dr.ctypes.data), C.c_void_p(Dc.ctypes.data)))
        return Dr, Dc

    def scaled_values(self, from_transpose=False):
        v = np.full(self.nnz, np.nan)
        _check(self.lib.uc_lp_get_scaled_values(self._h, int(bool(from_transpose)), C.c_void_p(v.ctypes.data)))
        return v

    def spmv(self, v, transpose=False):
        nin, nout = (self.m, self.n) if transpose else (self.n, self.m)
        va, vp = _host(v, np.float64)
        assert va.shape == (nin,)
        if nin == 0:
            va = np.zeros(1); vp = C.c_void_p(va.ctypes.data)
        out = np.zeros(max(nout, 1))
        _check(self.lib.uc_lp_spmv(self._h, int(bool(transpose)), vp, C.c_void_p(out.ctypes.data)))
        return out[:nout]

    def spmv_static(self, v_device_ptr, out_device_ptr, transpose=False, stream=None) -> None:
        """uc_lp_spmv_static: the product of `spmv` for callers that must not allocate device memory (the intermediates
        sit in a fixed 2 MiB array inside the library; m + n is limited to SPMV_STATIC_MAX_DOUBLES).  Both arguments are
        device addresses (ints) of caller-owned float64 buffers on the handle's device; the kernels are enqueued on
        `stream` (None = the handle's stream) and the call does not wait for them.  See include/uc_pdhg.h."""
        _check(self.lib.uc_lp_spmv_static(self._h, int(bool(transpose)), C.c_void_p(int(v_device_ptr)), C.c_void_p(int(out_device_ptr)),
                                          C.c_void_p(int(stream)) if stream is not None else None))

    def solve(self, x0=None, y0=None, trace_attempts=0, trace_checks=0, want_xy=True, stream=None, **params) -> Solution:
        """uc_pdhg_solve: host buffers in and out (H2D / D2H inside the call)."""
        prm = default_params(**params)
        keep = []
        if x0 is not None:
            a, p = _host(x0, np.float64); keep.append(a); prm.x0 = p
        if y0 is not None:
            a, p = _host(y0, np.float64); keep.append(a); prm.y0 = p
        if stream is not None:
            prm.stream = C.c_void_p(int(stream))
        att = np.zeros(max(trace_attempts, 1), dtype=ATTEMPT_DTYPE)
        chk = np.zeros(max(trace_checks, 1), dtype=CHECK_DTYPE)
        if trace_attempts:
            prm.attempt_trace = C.c_void_p(att.ctypes.data); prm.attempt_trace_cap = trace_attempts
        if trace_checks:
            prm.check_trace = C.c_void_p(chk.ctypes.data); prm.check_trace_cap = trace_checks
        x = np.zeros(self.n) if want_xy else None
        y = np.zeros(self.m) if want_xy else None
        res = Result()
        _check(self.lib.uc_pdhg_solve(self._h, C.cast(C.byref(prm), C.c_void_p),
                                      C.c_void_p(x.ctypes.data) if want_xy and self.n else None,
                                      C.c_void_p(y.ctypes.data) if want_xy and self.m else None,
                                      C.cast(C.byref(res), C.c_void_p)))
        return self._solution(res, x, y, att, chk, trace_attempts, trace_checks)

    def solve_device(self, x_out=None, y_out=None, x0=None, y0=None, trace_attempts=0, trace_checks=0,
                     stream=None, **params) -> Solution:
        """uc_pdhg_solve_device: x_out / y_out / x0 / y0 are CUDA torch tensors (float64) on the handle's
        device; torch only owns the memory and supplies the stream."""
        prm = default_params(**params)

        def dptr(t, k):
            if t is None:
                return None
            assert t.is_cuda and t.is_contiguous() and str(t.dtype) == "torch.float64" and t.numel() == k
            return C.c_void_p(t.data_ptr())
        prm.x0 = dptr(x0, self.n)
        prm.y0 = dptr(y0, self.m)
        if stream is not None:
            prm.stream = C.c_void_p(int(stream))
        att = np.zeros(max(trace_attempts, 1), dtype=ATTEMPT_DTYPE)
        chk = np.zeros(max(trace_checks, 1), dtype=CHECK_DTYPE)
        if trace_attempts:
            prm.attempt_trace = C.c_void_p(att.ctypes.data); prm.attempt_trace_cap = trace_attempts
        if trace_checks:
            prm.check_trace = C.c_void_p(chk.ctypes.data); prm.check_trace_cap = trace_checks
        res = Result()
        _check(self.lib.uc_pdhg_solve_device(self._h, C.cast(C.byref(prm), C.c_void_p), dptr(x_out, self.n),
                                             dptr(y_out, self.m), C.cast(C.byref(res), C.c_void_p)))
        return self._solution(res, x_out, y_out, att, chk, trace_attempts, trace_checks)

    @staticmethod
    def _solution(res, x, y, att, chk, na, nc):
        return Solution(x=x, y=y, status=res.status, returned_average=res.returned_average,
                        iterations=res.iterations, accepted=res.accepted, restarts=res.restarts,
                        rel_kkt=res.rel_kkt, rel_primal_res=res.rel_primal_res, rel_dual_res=res.rel_dual_res,
                        rel_gap=res.rel_gap, primal_obj=res.primal_obj, dual_obj=res.dual_obj, eta=res.eta,
                        omega=res.omega, solve_seconds=res.solve_seconds, loop_seconds=res.loop_seconds,
                        kernel_launches=res.kernel_launches,
                        attempts=att[:min(na, res.attempt_records)], checks=chk[:min(nc, res.check_records)])
