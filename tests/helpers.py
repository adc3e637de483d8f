"""Test-side references that are independent of both the oracle and the CUDA path:
brute-force vertex enumeration, a HiGHS wrapper, dense numpy KKT checks, golden readers."""
from __future__ import annotations

import itertools
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden_rows(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append(line.split())
    return rows


def vertex_enumeration(lp, tol=1e-9):
    """Exact LP optimum for tiny LPs: try every choice of n active constraints among rows and
    finite bounds (all 'E' rows always active), keep feasible points, return (best_obj, best_x)."""
    A = lp.dense().reshape(lp.m, lp.n)
    n, m = lp.n, lp.m
    eq = [i for i in range(m) if lp.sense[i] == ord("E")]
    ge = [i for i in range(m) if lp.sense[i] == ord("G")]
    cands = [("row", i) for i in ge]
    cands += [("lo", j) for j in range(n) if np.isfinite(lp.l[j])]
    cands += [("hi", j) for j in range(n) if np.isfinite(lp.u[j])]
    need = n - len(eq)
    best, best_x = np.inf, None
    if need < 0:
        return best, best_x
    for combo in itertools.combinations(cands, need):
        M = np.zeros((n, n)); r = np.zeros(n)
        k = 0
        for i in eq:
            M[k] = A[i]; r[k] = lp.b[i]; k += 1
        for kind, idx in combo:
            if kind == "row":
                M[k] = A[idx]; r[k] = lp.b[idx]
            else:
                M[k, idx] = 1.0; r[k] = lp.l[idx] if kind == "lo" else lp.u[idx]
            k += 1
        if abs(np.linalg.det(M)) < 1e-12:
            continue
        x = np.linalg.solve(M, r)
        ax = A @ x if m else np.zeros(0)
        if np.any(x < lp.l - tol) or np.any(x > lp.u + tol):
            continue
        if any(abs(ax[i] - lp.b[i]) > tol for i in eq) or any(ax[i] < lp.b[i] - tol for i in ge):
            continue
        obj = float(lp.c @ x)
        if obj < best - 1e-13:
            best, best_x = obj, x
    return best, best_x


def highs(lp):
    """scipy HiGHS solve.  Returns (objective, x, y) with y in the sign convention of the ABI:
    Lagrangian c'x - y'(Kx - q), so y_i >= 0 on 'G' rows."""
    from scipy.optimize import linprog
    A = lp.to_scipy()
    E = lp.sense == ord("E")
    G = ~E
    bounds = [(None if np.isinf(a) else a, None if np.isinf(b) else b) for a, b in zip(lp.l, lp.u)]
    kw = {}
    if G.any():
        kw.update(A_ub=-A[G], b_ub=-lp.b[G])
    if E.any():
        kw.update(A_eq=A[E], b_eq=lp.b[E])
    r = linprog(lp.c, bounds=bounds, method="highs", **kw)
    assert r.status == 0, r.message
    y = np.zeros(lp.m)
    if E.any():
        y[E] = r.eqlin.marginals            # d obj / d b_eq
    if G.any():
        y[G] = -r.ineqlin.marginals         # rows were negated: d obj / d(-b) = -(d obj / d b)
    return float(r.fun), np.asarray(r.x), y


def dense_kkt(lp, x, y):
    """KKT quantities of (x, y) from dense numpy algebra -- a second, independent statement of
    DESIGN.md R9: returns dict(rp, rd, pobj, dobj, lam)."""
    A = lp.dense().reshape(lp.m, lp.n)
    a = A @ x - lp.b
    rp = np.where(lp.sense == ord("E"), a, np.minimum(a, 0.0))
    rho = lp.c - A.T @ y
    lam = np.maximum(rho, 0.0) * np.isfinite(lp.l) + np.minimum(rho, 0.0) * np.isfinite(lp.u)
    rd = rho - lam
    lo = np.where(np.isfinite(lp.l), lp.l, 0.0)
    hi = np.where(np.isfinite(lp.u), lp.u, 0.0)
    dobj = lp.b @ y + lo @ np.maximum(lam, 0.0) + hi @ np.minimum(lam, 0.0)
    return dict(rp=np.linalg.norm(rp), rd=np.linalg.norm(rd), pobj=float(lp.c @ x), dobj=float(dobj),
                lam=lam, slack=a)


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(b), 1e-300))
