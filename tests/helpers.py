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


def restart_replay(lp, sol, vs, beta_s=0.2, beta_n=0.8, beta_a=0.36, theta=0.5):
    """Independent numpy restatement of DESIGN.md R9..R11 (restart decision and primal weight), fed ONLY with
    iterates: `sol` is an oracle Solution with dump_checks (scaled current iterate, scaled average and w at every
    check), `vs` the scaled matrix values K~ (pinned separately by the preconditioner tests).  Everything else is
    recomputed here with dense algebra: the scaled data, omega0, KKT_omega of current / average / restart point,
    candidate, restart kind, and the primal weight in its closed form
        omega_new = (Dy / Dx)^theta * omega_old^(1 - theta)     (= sqrt(omega_old * Dy / Dx), the geometric mean, for
                                                                 the default theta = 1/2).
    Returns a list of dicts, one per check."""
    m, n = lp.m, lp.n
    Kt = np.zeros((m, n))
    rows = np.repeat(np.arange(m), np.diff(lp.row_ptr))
    Kt[rows, lp.col_idx] = vs
    Dr, Dc = sol.Dr, sol.Dc
    with np.errstate(invalid="ignore"):
        c, q = lp.c / Dc, lp.b / Dr
        l = np.where(lp.l <= -1e20, -np.inf, lp.l * Dc)
        u = np.where(lp.u >= 1e20, np.inf, lp.u * Dc)
    isE = lp.sense == ord("E")

    def kkt_omega(x, y, omega):
        a = Kt @ x - q
        rp = np.where(isE, a, np.minimum(a, 0.0))
        rho = c - Kt.T @ y
        lam = np.maximum(rho, 0.0) * np.isfinite(l) + np.minimum(rho, 0.0) * np.isfinite(u)
        rd = rho - lam
        lo = np.where(np.isfinite(l), l, 0.0); hi = np.where(np.isfinite(u), u, 0.0)
        dobj = q @ y + lo @ np.maximum(lam, 0.0) + hi @ np.minimum(lam, 0.0)
        gap = c @ x - dobj
        return float(np.sqrt(omega ** 2 * (rp @ rp) + (rd @ rd) / omega ** 2 + gap ** 2))

    nc, nq = np.linalg.norm(c), np.linalg.norm(q)
    omega = nc / nq if (nc > 1e-10 and nq > 1e-10) else 1.0
    xr, yr = np.clip(np.zeros(n), l, u), np.zeros(m)
    t0, mu_prev = 0, np.inf
    out = []
    for i, rec in enumerate(sol.checks[:len(sol.check_w)]):
        k = int(rec["k"])
        xc, yc, xa, ya, w = sol.check_x[i], sol.check_y[i], sol.check_avg_x[i], sol.check_avg_y[i], sol.check_w[i]
        k_cur = kkt_omega(xc, yc, omega)
        k_avg = kkt_omega(xa, ya, omega) if w > 0 else np.inf
        cand = int(w > 0 and k_avg < k_cur)
        zc = (xa, ya) if cand else (xc, yc)
        mu_c, mu_r = (k_avg if cand else k_cur), kkt_omega(xr, yr, omega)
        t = k - t0
        kind = 0
        if mu_c <= beta_s * mu_r:
            kind = 1
        elif mu_c <= beta_n * mu_r and mu_c > mu_prev:
            kind = 2
        elif t >= beta_a * k:
            kind = 3
        d = dict(k=k, kkt_cur=k_cur, kkt_avg=k_avg, candidate=cand, mu_c=mu_c, mu_r=mu_r, mu_prev=mu_prev, t=t,
                 kind=kind, omega_before=omega, Dx=None, Dy=None)
        if kind:
            Dx, Dy = float(np.linalg.norm(zc[0] - xr)), float(np.linalg.norm(zc[1] - yr))
            if Dx > 1e-10 and Dy > 1e-10:
                omega = float(np.sqrt(omega * Dy / Dx)) if theta == 0.5 else float((Dy / Dx) ** theta * omega ** (1.0 - theta))
            xr, yr = zc[0].copy(), zc[1].copy()
            t0, mu_prev = k, np.inf
            d.update(Dx=Dx, Dy=Dy)
        else:
            mu_prev = mu_c
        d["omega_after"] = omega
        out.append(d)
    return out
