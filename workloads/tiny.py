"""Tiny hand-checkable LPs used as pins (data only; expected values live in the tests).

Each builder cites where its expected answer comes from (SURVEY.md 8(c) "Pins").
"""
from __future__ import annotations

import numpy as np

from .lp import LP, from_dense

INF = np.inf


def one_by_one(l: float = 0.0, u: float = 10.0) -> LP:
    """min x s.t. x >= 1, l <= x <= u; default 0 <= x <= 10 (SURVEY 8(c) worked PDHG-step example; x*=1, y*=1).
    (l, u) = (-inf, inf) is the free-variable case of the worked restart example (tests/golden/restart_1x1.txt)."""
    return from_dense([[1.0]], ["G"], [1.0], [1.0], [l], [u], name="one_by_one")


def two_var() -> LP:
    """min -x1 - 2 x2 s.t. -x1 - x2 >= -4, 0 <= x <= 3: x*=(1,3), obj -7, y*=1."""
    return from_dense([[-1.0, -1.0]], ["G"], [-4.0], [-1.0, -2.0], [0.0, 0.0], [3.0, 3.0], name="two_var")


def precond_2x2() -> LP:
    """K = [[4, 1], [0, 0.25]] (SURVEY 8(c) worked preconditioner example)."""
    return from_dense([[4.0, 1.0], [0.0, 0.25]], ["E", "E"], [1.0, 1.0], [1.0, 1.0],
                      [0.0, 0.0], [10.0, 10.0], name="precond_2x2")


def box_only(n: int = 7, seed: int = 0, with_rows: int = 0) -> LP:
    """Box-only LP (m = 0, or `with_rows` all-zero rows 0 >= -1): x_j = l_j if c_j > 0, u_j if c_j < 0."""
    rng = np.random.default_rng(seed)
    c = rng.standard_normal(n)
    c[0] = 0.0
    l = -rng.uniform(0.5, 3.0, n)
    u = rng.uniform(0.5, 3.0, n)
    m = with_rows
    return LP(m=m, n=n, row_ptr=np.zeros(m + 1, np.int64), col_idx=np.zeros(0, np.int32),
              val=np.zeros(0), sense=np.full(m, ord("G"), np.uint8), b=-np.ones(m), c=c, l=l, u=u,
              name=f"box_only_n{n}")


def economic_dispatch(G: int = 6, seed: int = 0, demand_frac: float = 0.55):
    """Single-bus, single-period economic dispatch with commitment fixed to 1 and Pmin = 0:
        min sum cost_g p_g  s.t.  sum p_g = d,  0 <= p_g <= Pmax_g.
    Optimum = merit order (north_star: 'single-bus economic dispatch equals the merit-order
    solution'); the balance dual is the marginal unit's cost.  Returns (lp, pmax, cost, d)."""
    rng = np.random.default_rng(seed)
    pmax = rng.uniform(0.2, 5.0, G)
    cost = rng.uniform(10.0, 80.0, G)
    d = demand_frac * pmax.sum()
    lp = from_dense(np.ones((1, G)), ["E"], [d], cost, np.zeros(G), pmax, name=f"dispatch_G{G}")
    return lp, pmax, cost, d


def small_random(n: int, m: int, seed: int, density: float = 0.7) -> LP:
    """Feasible, bounded random LP with n <= 8 variables for brute-force vertex enumeration."""
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((m, n)) * (rng.uniform(size=(m, n)) < density)
    for i in range(m):                      # no empty rows
        if not A[i].any():
            A[i, rng.integers(0, n)] = 1.0
    l = -rng.uniform(0.0, 2.0, n)
    u = rng.uniform(0.5, 3.0, n)
    x0 = l + rng.uniform(0.1, 0.9, n) * (u - l)
    sense = ["E" if (i % 3 == 0) else "G" for i in range(m)]
    slack = rng.uniform(0.0, 1.0, m) * np.array([0.0 if s == "E" else 1.0 for s in sense])
    b = A @ x0 - slack
    c = rng.standard_normal(n)
    return from_dense(A, sense, b, c, l, u, name=f"small_n{n}_m{m}_s{seed}")


def free_var_lp() -> LP:
    """LP with a free variable and a one-sided variable (exercises infinite bounds):
        min x1 + 2 x2 + 0 x3  s.t.  x1 + x3 = 2,  x2 - x3 >= -1,  x1 in [0, inf), x2 in [0, inf), x3 free.
    Substituting x1 = 2 - x3 >= 0, x2 >= max(0, x3 - 1): obj = 2 - x3 + 2 max(0, x3 - 1) is minimised
    on x3 in [1, 2]... strictly: at x3 = 1 the slope changes from -1 to +1, so x* = (1, 0, 1), obj = 1."""
    return from_dense([[1.0, 0.0, 1.0], [0.0, 1.0, -1.0]], ["E", "G"], [2.0, -1.0], [1.0, 2.0, 0.0],
                      [0.0, 0.0, -INF], [INF, INF, INF], name="free_var")
