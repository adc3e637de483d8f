"""TEST INFRASTRUCTURE -- ctypes front end of oracle/pdhg_oracle.c (the CPU fp64 oracle).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2607_03627_b200 and shares no code with it.
Argument marshalling only; all arithmetic is in the C file (which cites DESIGN.md's readings).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pdhg_oracle.c")
# PDHG_ORACLE_LIB: load another build of the same source instead (the -fsanitize=address,undefined build of
# profiles/r03_oracle_sanitizers.md); it is never built or rebuilt from here
_LIB = os.environ.get("PDHG_ORACLE_LIB") or os.path.join(_HERE, "libpdhg_oracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-shared", "-fPIC", "-Wall"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (single thread, no FMA contraction)."""
    if os.environ.get("PDHG_ORACLE_LIB"):
        return _LIB
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Params(C.Structure):
    _fields_ = [("iter_limit", C.c_int64), ("eps_rel", C.c_double), ("eps_abs", C.c_double),
                ("check_every", C.c_int32), ("ruiz_iters", C.c_int32), ("pc_alpha", C.c_double),
                ("fixed_iterations", C.c_int64), ("beta_sufficient", C.c_double),
                ("beta_necessary", C.c_double), ("beta_artificial", C.c_double),
                ("weight_smoothing", C.c_double), ("restarts_enabled", C.c_int32), ("pad_", C.c_int32),
                ("frozen_eta", C.c_double), ("eta0", C.c_double), ("omega0", C.c_double)]


class Result(C.Structure):
    _fields_ = [("status", C.c_int32), ("returned_average", C.c_int32), ("iterations", C.c_int64),
                ("accepted", C.c_int64), ("restarts", C.c_int64), ("rel_kkt", C.c_double),
                ("rel_primal_res", C.c_double), ("rel_dual_res", C.c_double), ("rel_gap", C.c_double),
                ("primal_obj", C.c_double), ("dual_obj", C.c_double), ("eta", C.c_double), ("omega", C.c_double)]


ATTEMPT_DTYPE = np.dtype([("eta_used", "f8"), ("eta_bar", "f8"), ("eta_next", "f8"), ("dx2", "f8"),
                          ("dy2", "f8"), ("inter", "f8"), ("accepted", "i4"), ("pad_", "i4")])
CHECK_DTYPE = np.dtype([("k", "i8"), ("restart_kind", "i4"), ("candidate", "i4"), ("omega_after", "f8"),
                        ("mu_c", "f8"), ("mu_r", "f8"), ("relkkt_cur", "f8"), ("relkkt_avg", "f8")])

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_pdhg_solve.restype = C.c_int
    return _lib


def _p(a, typ=C.c_double):
    return None if a is None else a.ctypes.data_as(C.POINTER(typ))


def default_params(**kw) -> Params:
    p = Params()
    lib().oracle_default_params(C.byref(p))
    for k, v in kw.items():
        assert hasattr(p, k), k
        setattr(p, k, v)
    return p


@dataclass
class Solution:
    x: np.ndarray
    y: np.ndarray
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
    attempts: np.ndarray
    checks: np.ndarray
    dump_x: np.ndarray | None
    dump_y: np.ndarray | None
    avg_x: np.ndarray
    avg_y: np.ndarray
    avg_w: float
    Dr: np.ndarray
    Dc: np.ndarray
    check_x: np.ndarray | None = None      # [checks, n] scaled current iterate as each check saw it
    check_y: np.ndarray | None = None
    check_avg_x: np.ndarray | None = None  # [checks, n] scaled average at each check (current iterate if w = 0)
    check_avg_y: np.ndarray | None = None
    check_w: np.ndarray | None = None      # [checks] weight sum w at each check


def _csr(lp):
    return (C.c_int64(lp.m), C.c_int64(lp.n), _p(lp.row_ptr, C.c_int64), _p(lp.col_idx, C.c_int32), _p(lp.val))


def solve(lp, x0=None, y0=None, trace_attempts=0, trace_checks=4096, dump=0, dump_checks=0, **params) -> Solution:
    """Run the oracle on `lp` (a workloads.LP).  Keyword params override oracle_default_params."""
    prm = default_params(**params)
    m, n = lp.m, lp.n
    x = np.zeros(n); y = np.zeros(m)
    att = np.zeros(max(trace_attempts, 1), dtype=ATTEMPT_DTYPE)
    chk = np.zeros(max(trace_checks, 1), dtype=CHECK_DTYPE)
    na, nc = C.c_int64(0), C.c_int64(0)
    dx = np.zeros((dump, n)) if dump else None
    dy = np.zeros((dump, m)) if dump else None
    ax = np.zeros(n); ay = np.zeros(m); aw = C.c_double(0.0)
    Dr = np.zeros(m); Dc = np.zeros(n)
    cx = np.zeros((dump_checks, n)) if dump_checks else None
    cy = np.zeros((dump_checks, m)) if dump_checks else None
    cax = np.zeros((dump_checks, n)) if dump_checks else None
    cay = np.zeros((dump_checks, m)) if dump_checks else None
    cw = np.zeros(dump_checks) if dump_checks else None
    res = Result()
    x0 = None if x0 is None else np.ascontiguousarray(x0, dtype=np.float64)
    y0 = None if y0 is None else np.ascontiguousarray(y0, dtype=np.float64)
    rc = lib().oracle_pdhg_solve(*_csr(lp), _p(lp.sense, C.c_ubyte), _p(lp.b), _p(lp.c), _p(lp.l), _p(lp.u),
                                 C.byref(prm), _p(x0), _p(y0), _p(x), _p(y), C.byref(res),
                                 C.c_void_p(att.ctypes.data), C.c_int64(trace_attempts), C.byref(na),
                                 C.c_void_p(chk.ctypes.data), C.c_int64(trace_checks), C.byref(nc),
                                 _p(dx), _p(dy), C.c_int64(dump), _p(ax), _p(ay), C.byref(aw), _p(Dr), _p(Dc),
                                 _p(cx), _p(cy), _p(cax), _p(cay), _p(cw), C.c_int64(dump_checks))
    if rc != 0:
        raise ValueError(f"oracle_pdhg_solve returned {rc}")
    return Solution(x=x, y=y, status=res.status, returned_average=res.returned_average,
                    iterations=res.iterations, accepted=res.accepted, restarts=res.restarts,
                    rel_kkt=res.rel_kkt, rel_primal_res=res.rel_primal_res, rel_dual_res=res.rel_dual_res,
                    rel_gap=res.rel_gap, primal_obj=res.primal_obj, dual_obj=res.dual_obj, eta=res.eta,
                    omega=res.omega, attempts=att[:min(na.value, trace_attempts)],
                    checks=chk[:min(nc.value, trace_checks)], dump_x=dx, dump_y=dy,
                    avg_x=ax, avg_y=ay, avg_w=aw.value, Dr=Dr, Dc=Dc,
                    check_x=None if cx is None else cx[:min(nc.value, dump_checks)],
                    check_y=None if cy is None else cy[:min(nc.value, dump_checks)],
                    check_avg_x=None if cax is None else cax[:min(nc.value, dump_checks)],
                    check_avg_y=None if cay is None else cay[:min(nc.value, dump_checks)],
                    check_w=None if cw is None else cw[:min(nc.value, dump_checks)])


def precondition(lp, ruiz_iters=10, pc_alpha=1.0):
    """(val_scaled, Dr, Dc) with K = diag(Dr) Ktilde diag(Dc)   (R1)."""
    vs = np.zeros(lp.nnz); Dr = np.zeros(lp.m); Dc = np.zeros(lp.n)
    lib().oracle_precondition(*_csr(lp), C.c_int32(ruiz_iters), C.c_double(pc_alpha), _p(vs), _p(Dr), _p(Dc))
    return vs, Dr, Dc


def spmv(lp, v, val=None):
    out = np.zeros(lp.m)
    val = lp.val if val is None else val
    v = np.ascontiguousarray(v, dtype=np.float64)
    lib().oracle_spmv(C.c_int64(lp.m), _p(lp.row_ptr, C.c_int64), _p(lp.col_idx, C.c_int32), _p(val), _p(v), _p(out))
    return out


def spmv_t(lp, y, val=None):
    out = np.zeros(lp.n)
    val = lp.val if val is None else val
    y = np.ascontiguousarray(y, dtype=np.float64)
    lib().oracle_spmv_t(C.c_int64(lp.m), C.c_int64(lp.n), _p(lp.row_ptr, C.c_int64), _p(lp.col_idx, C.c_int32),
                        _p(val), _p(y), _p(out))
    return out


def kkt_unscaled(lp, x, y):
    """dict(rp, rd, pobj, dobj, rel_kkt) of an ORIGINAL-space point, straight from the LP's definition."""
    out = np.zeros(5)
    x = np.ascontiguousarray(x, dtype=np.float64); y = np.ascontiguousarray(y, dtype=np.float64)
    lib().oracle_kkt_unscaled(*_csr(lp), _p(lp.sense, C.c_ubyte), _p(lp.b), _p(lp.c), _p(lp.l), _p(lp.u),
                              _p(x), _p(y), _p(out))
    return dict(rp=out[0], rd=out[1], pobj=out[2], dobj=out[3], rel_kkt=out[4])
