"""The hand derivation behind tests/golden/restart_1x1.txt, in executable form.

It calls NEITHER oracle/ NOR the CUDA path: it is the arithmetic of DESIGN.md "Worked restart example" written
with plain Python floats for the case m = n = 1, K = [1], where every vector of readings R2..R11 is one number,
every norm an absolute value and every SpMV a multiplication -- so that each printed line can be checked with a
pocket calculator against the formulas of DESIGN.md (R3..R5 for an attempt, R9 for the KKT terms, R10 for the
restart decision, R11 for the primal weight).  DESIGN.md carries the first lines out by hand.

LPs:  min x  s.t.  x >= 1  ('G' row),  l <= x <= u,  with  (l, u) = (-inf, +inf)  ["free"]  and  (0, 10)  ["bounded"];
no preconditioning (it is the identity on K = [1]), x0 = y0 = 0, eta0 = 1 / max|K| = 1, omega0 = |c| / |q| = 1,
a check after EVERY attempt (check_every = 1).

    python tests/golden/restart_1x1_derivation.py  >  tests/golden/restart_1x1.txt
"""
import math

INF = math.inf
BETA_S, BETA_N, BETA_A, THETA = 0.2, 0.8, 0.36, 0.5
C, Q = 1.0, 1.0


def kkt_terms(x, y, l, u):
    """R9 for one variable and one 'G' row: (r_p^2, r_d^2, pobj, dobj)."""
    a = x - Q
    rp = min(a, 0.0)                                  # 'G' row: only a violation counts
    rho = C - y
    lam = 0.0
    if rho > 0.0 and l > -INF:
        lam = rho                                     # reduced cost absorbed by the finite lower bound
    if rho < 0.0 and u < INF:
        lam = rho                                     # ... by the finite upper bound
    rd = rho - lam
    dobj = Q * y + (l * lam if lam > 0.0 else (u * lam if lam < 0.0 else 0.0))
    return rp * rp, rd * rd, C * x, dobj


def kkt_omega(t, omega):
    rp2, rd2, pobj, dobj = t
    return math.sqrt(omega * omega * rp2 + rd2 / (omega * omega) + (pobj - dobj) ** 2)


def derive(name, l, u, attempts):
    x, y = min(max(0.0, l), u), 0.0                   # R2
    eta, omega = 1.0, 1.0
    k, t0, w, xs, ys, mu_prev = 0, 0, 0.0, 0.0, 0.0, INF
    xr, yr, Tr = x, y, kkt_terms(x, y, l, u)
    print(f"# ---- {name}: l = {l}, u = {u}")
    print("# A k  x_trial        y_trial        eta_used       eta_bar        accepted  eta_next")
    print("# C k  kkt_cur        kkt_avg        candidate  mu_c           mu_r           t   kind  omega_after    x_after        y_after")
    while k < attempts:
        k += 1                                        # R3..R6: one attempt
        tau, sig = eta / omega, eta * omega
        xn = min(max(x - tau * (C - y), l), u)
        xbar = 2.0 * xn - x
        yn = max(y + sig * (Q - xbar), 0.0)
        dx, dy = xn - x, yn - y
        N, inter = omega * dx * dx + dy * dy / omega, abs(dy * dx)
        eta_bar = N / (2.0 * inter) if inter > 0.0 else INF
        grow = (1.0 + (k + 1) ** -0.6) * eta
        eta_next = grow if eta_bar == INF else min((1.0 - (k + 1) ** -0.3) * eta_bar, grow)
        accept = eta <= eta_bar
        print(f"{name} A {k:<2d} {xn:<14.10g} {yn:<14.10g} {eta:<14.10g} {eta_bar:<14.10g} {int(accept):<9d} {eta_next:.10g}")
        if accept:
            x, y = xn, yn
            xs += eta * xn; ys += eta * yn; w += eta
        eta = eta_next
        # R8..R11: the check (check_every = 1)
        Tc = kkt_terms(x, y, l, u)
        have_avg = w > 0.0
        Ta = kkt_terms(xs / w, ys / w, l, u) if have_avg else Tc
        kc, ka = kkt_omega(Tc, omega), kkt_omega(Ta, omega)
        cand = 1 if (have_avg and ka < kc) else 0     # strict <: a tie keeps the current iterate
        Tk = Ta if cand else Tc
        mu_c, mu_r, t = kkt_omega(Tk, omega), kkt_omega(Tr, omega), k - t0
        kind = 0
        if mu_c <= BETA_S * mu_r:
            kind = 1                                  # sufficient decay
        elif mu_c <= BETA_N * mu_r and mu_c > mu_prev:
            kind = 2                                  # necessary decay + no longer improving
        elif t >= BETA_A * k:
            kind = 3                                  # artificial
        if kind:
            xc, yc = (xs / w, ys / w) if cand else (x, y)
            Dx, Dy = abs(xc - xr), abs(yc - yr)
            if Dx > 1e-10 and Dy > 1e-10:
                omega = math.exp(THETA * math.log(Dy / Dx) + (1.0 - THETA) * math.log(omega))
            x, y, xr, yr, Tr = xc, yc, xc, yc, Tk
            xs = ys = w = 0.0
            t0, mu_prev = k, INF
        else:
            mu_prev = mu_c
        print(f"{name} C {k:<2d} {kc:<14.10g} {ka:<14.10g} {cand:<10d} {mu_c:<14.10g} {mu_r:<14.10g} {t:<3d} {kind:<5d} {omega:<14.10g} {x:<14.10g} {y:.10g}")


if __name__ == "__main__":
    print("# Worked restart example (DESIGN.md 'Worked restart example'; readings R9, R10, R11): two 1x1 LPs,")
    print("#   min x s.t. x >= 1, l <= x <= u,  K = [1], no preconditioning, x0 = y0 = 0, eta0 = 1, omega0 = 1, check_every = 1.")
    print("# Written by tests/golden/restart_1x1_derivation.py (plain scalar arithmetic; calls neither oracle/ nor the")
    print("# CUDA path); the first lines are carried out by hand in DESIGN.md.  10 significant digits.")
    print("# 'A' lines: one attempt (trial point, step size used, bound eta_bar, accept flag, next step size).")
    print("# 'C' lines: the check after it (KKT_omega of current and average with the omega BEFORE the check, candidate")
    print("#   0 = current / 1 = average, mu_c, mu_r, t = k - t0, restart kind 0 none / 1 sufficient / 2 necessary /")
    print("#   3 artificial, omega after the check, and the iterate the next attempt starts from).")
    derive("free", -INF, INF, 13)
    derive("bounded", 0.0, 10.0, 13)
