"""Pins for the CPU oracle (no GPU): each test checks oracle/ against something OTHER than itself --
values printed in SURVEY.md 8(c) worked examples (tests/golden/), closed forms, brute-force vertex
enumeration, HiGHS, dense numpy algebra, and textbook invariants of PDHG.  DESIGN.md lists which
reading (R1..R14) each pin covers; none remains 'parity unpinned' (R10 / R11: the worked restart example and the
dense replay of every restart decision below)."""
import math

import numpy as np
import pytest

import oracle
from workloads import tiny, uc_config, fix_commitment
from workloads.lp import from_dense

from helpers import read_golden_rows, vertex_enumeration, highs, dense_kkt, rel_l2, restart_replay


def _f(s):
    return float(s)


# ------------------------------------------------------------------ R2..R6: the PDHG step
def test_worked_1x1_step_example_matches_golden():
    rows = read_golden_rows("pdhg_step_1x1.txt")
    lp = tiny.one_by_one()
    s = oracle.solve(lp, fixed_iterations=len(rows), ruiz_iters=0, pc_alpha=0.0,
                     trace_attempts=len(rows), dump=len(rows))
    x_cur, y_cur = 0.0, 0.0
    eta = 1.0
    for r, a, xd, yd in zip(rows, s.attempts, s.dump_x[:, 0], s.dump_y[:, 0]):
        k, x_new, y_new, eta_bar, acc, eta_next = int(r[0]), _f(r[1]), _f(r[2]), _f(r[3]), int(r[4]), _f(r[5])
        assert a["eta_used"] == pytest.approx(eta, rel=2e-9)
        assert a["accepted"] == acc, f"attempt {k}"
        if not math.isnan(eta_bar):
            assert a["eta_bar"] == pytest.approx(eta_bar, rel=2e-9)
        assert a["eta_next"] == pytest.approx(eta_next, rel=2e-9)
        if acc:
            x_cur, y_cur = x_new, y_new
        assert xd == pytest.approx(x_cur, rel=2e-9, abs=1e-12)      # iterate after attempt k
        assert yd == pytest.approx(y_cur, rel=2e-9, abs=1e-12)
        eta = eta_next
    # limit point of the same example: x*=1, y*=1, objective 1
    s = oracle.solve(lp, eps_rel=1e-10, eps_abs=1e-10, ruiz_iters=0, pc_alpha=0.0)
    assert s.status == 0 and s.x[0] == pytest.approx(1.0, abs=1e-8) and s.y[0] == pytest.approx(1.0, abs=1e-8)


def test_step_first_attempts_by_hand():
    """k=1..3 of the 1x1 example re-derived here from the update formulas with plain floats."""
    lp = tiny.one_by_one()
    s = oracle.solve(lp, fixed_iterations=3, ruiz_iters=0, pc_alpha=0.0, trace_attempts=3)
    e1 = 1.0 + 2.0 ** -0.6                      # k=1: x'=0, y'=1, eta_bar=inf -> grow
    e2 = (1.0 + 3.0 ** -0.6) * e1               # k=2: x'=0, y'=1+e1
    y2 = 1.0 + e1
    x3 = e2 * (y2 - 1.0)                        # k=3: x' = 0 - e2 (1 - y2)
    dy = -y2                                    # y' = max(y2 + e2 (1 - 2 x3), 0) = 0
    ebar3 = (x3 * x3 + dy * dy) / (2.0 * abs(dy * x3))
    e3 = (1.0 - 4.0 ** -0.3) * ebar3
    assert y2 + e2 * (1 - 2 * x3) < 0
    assert s.attempts["eta_next"][0] == pytest.approx(e1, rel=1e-14)
    assert s.attempts["eta_next"][1] == pytest.approx(e2, rel=1e-14)
    assert s.attempts["eta_bar"][2] == pytest.approx(ebar3, rel=1e-14)
    assert s.attempts["accepted"].tolist() == [1, 1, 0]
    assert s.attempts["eta_next"][2] == pytest.approx(e3, rel=1e-14)


# ------------------------------------------------------------------ R1: preconditioning
def test_worked_2x2_preconditioner_matches_golden():
    g = {r[0]: np.array([float(v) for v in r[1:]]) for r in read_golden_rows("precond_2x2.txt")}
    lp = tiny.precond_2x2()
    vs, Dr, Dc = oracle.precondition(lp, ruiz_iters=10, pc_alpha=0.0)
    np.testing.assert_allclose(Dr, g["ruiz_Dr"], rtol=2e-10)
    np.testing.assert_allclose(Dc, g["ruiz_Dc"], rtol=2e-10)
    np.testing.assert_allclose(vs, g["ruiz_K"], rtol=2e-10)
    vs2, _, _ = oracle.precondition(lp, ruiz_iters=2, pc_alpha=0.0)     # passes 3..10 change nothing
    np.testing.assert_allclose(vs2, vs, rtol=1e-15)
    vs, Dr, Dc = oracle.precondition(lp, ruiz_iters=10, pc_alpha=1.0)
    np.testing.assert_allclose(Dr, g["final_Dr"], rtol=2e-10)
    np.testing.assert_allclose(Dc, g["final_Dc"], rtol=2e-10)
    np.testing.assert_allclose(vs, g["final_K"], rtol=2e-10)
    Kt = np.array([[vs[0], vs[1]], [0.0, vs[2]]])
    assert np.linalg.svd(Kt, compute_uv=False)[0] == pytest.approx(1.0, abs=1e-12)


def test_ruiz_on_diagonal_matrix_closed_form():
    a = np.array([4.0, -9.0, 0.25, 1e-4, -1e4])
    lp = from_dense(np.diag(a), ["E"] * 5, np.ones(5), np.ones(5), -np.ones(5), np.ones(5))
    for iters in (1, 10):
        vs, Dr, Dc = oracle.precondition(lp, ruiz_iters=iters, pc_alpha=0.0)
        np.testing.assert_allclose(Dr, np.sqrt(np.abs(a)), rtol=1e-15)
        np.testing.assert_allclose(Dc, np.sqrt(np.abs(a)), rtol=1e-15)
        np.testing.assert_allclose(vs, np.sign(a), rtol=1e-15)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_preconditioner_identities_and_operator_norm(seed):
    lp = tiny.small_random(8, 6, seed, density=0.6)
    vs, Dr, Dc = oracle.precondition(lp)
    K = lp.dense()
    Kt = np.zeros_like(K)
    rows = np.repeat(np.arange(lp.m), np.diff(lp.row_ptr))
    Kt[rows, lp.col_idx] = vs
    np.testing.assert_allclose(Kt * Dr[:, None] * Dc[None, :], K, rtol=4e-15, atol=0)     # K = Dr Kt Dc
    assert np.linalg.svd(Kt, compute_uv=False)[0] <= 1.0 + 1e-12                          # Pock-Chambolle lemma
    # Ruiz alone equilibrates: row and column inf-norms approach 1, monotonically
    dev_prev = np.inf
    for it in (1, 3, 10):
        vr, _, _ = oracle.precondition(lp, ruiz_iters=it, pc_alpha=0.0)
        Kr = np.zeros_like(K); Kr[rows, lp.col_idx] = vr
        dev = max(np.abs(np.abs(Kr).max(axis=1) - 1).max(), np.abs(np.abs(Kr).max(axis=0) - 1).max())
        assert dev <= dev_prev + 1e-15
        dev_prev = dev
    assert dev_prev < 0.05


def test_preconditioner_on_uc_config0_operator_norm_and_empty_handling():
    import scipy.sparse as sp
    import scipy.sparse.linalg as spl
    lp = uc_config(0)
    vs, Dr, Dc = oracle.precondition(lp)
    Kt = sp.csr_matrix((vs, lp.col_idx, lp.row_ptr), shape=(lp.m, lp.n))
    smax = spl.svds(Kt, k=1, return_singular_vectors=False)[0]
    assert smax <= 1.0 + 1e-10
    assert np.all(Dr > 0) and np.all(Dc > 0) and np.all(np.isfinite(Dr)) and np.all(np.isfinite(Dc))
    # an LP with an empty row and an empty column: scaling factor 1 there
    lp2 = from_dense([[2.0, 0.0, 0.0], [0.0, 0.0, 0.0]], ["G", "G"], [0.0, -1.0], [1.0, 1.0, 1.0],
                     [0.0] * 3, [1.0] * 3)
    _, Dr2, Dc2 = oracle.precondition(lp2)
    assert Dr2[1] == 1.0 and Dc2[1] == 1.0 and Dc2[2] == 1.0


# ------------------------------------------------------------------ SpMV pair
def test_spmv_pair_dense_and_adjoint():
    rng = np.random.default_rng(5)
    lp = tiny.small_random(8, 6, 3)
    K = lp.dense()
    x = rng.standard_normal(lp.n); y = rng.standard_normal(lp.m)
    np.testing.assert_allclose(oracle.spmv(lp, x), K @ x, rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(oracle.spmv_t(lp, y), K.T @ y, rtol=1e-14, atol=1e-15)
    lp = uc_config(0)
    x = rng.standard_normal(lp.n); y = rng.standard_normal(lp.m)
    lhs, rhs = y @ oracle.spmv(lp, x), oracle.spmv_t(lp, y) @ x
    assert abs(lhs - rhs) <= 1e-13 * max(abs(lhs), 1.0) * 10
    np.testing.assert_allclose(oracle.spmv(lp, x), lp.to_scipy() @ x, rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(oracle.spmv_t(lp, y), lp.to_scipy().T @ y, rtol=1e-13, atol=1e-13)


# ------------------------------------------------------------------ closed forms
@pytest.mark.parametrize("rows", [0, 3])
def test_box_only_lp_closed_form(rows):
    lp = tiny.box_only(7, seed=1, with_rows=rows)
    s = oracle.solve(lp, eps_rel=1e-9, eps_abs=1e-9)
    expect = np.where(lp.c > 0, lp.l, np.where(lp.c < 0, lp.u, np.clip(0.0, lp.l, lp.u)))
    assert s.status == 0
    np.testing.assert_allclose(s.x, expect, atol=1e-9)
    assert s.primal_obj == pytest.approx(np.minimum(lp.c * lp.l, lp.c * lp.u).sum(), rel=1e-9)
    assert s.iterations <= 64 * 4                      # reached in finitely many attempts


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_single_bus_economic_dispatch_is_merit_order(seed):
    lp, pmax, cost, d = tiny.economic_dispatch(6, seed)
    order = np.argsort(cost)
    p = np.zeros(6); left = d; marginal = None
    for g in order:
        p[g] = min(pmax[g], left); left -= p[g]
        if marginal is None and left <= 1e-15:
            marginal = cost[g]
    s = oracle.solve(lp, eps_rel=1e-9, eps_abs=1e-9)
    assert s.status == 0
    np.testing.assert_allclose(s.x, p, atol=2e-6)
    assert s.primal_obj == pytest.approx(float(cost @ p), rel=1e-7)
    assert s.y[0] == pytest.approx(marginal, rel=1e-5)             # balance dual = marginal unit's cost


def test_worked_two_variable_lp():
    s = oracle.solve(tiny.two_var(), eps_rel=1e-10, eps_abs=1e-10)
    assert s.status == 0
    np.testing.assert_allclose(s.x, [1.0, 3.0], atol=1e-7)
    np.testing.assert_allclose(s.y, [1.0], atol=1e-7)
    assert s.primal_obj == pytest.approx(-7.0, abs=1e-7) and s.dual_obj == pytest.approx(-7.0, abs=1e-7)


def test_free_and_one_sided_variables():
    s = oracle.solve(tiny.free_var_lp(), eps_rel=1e-10, eps_abs=1e-10)
    assert s.status == 0
    np.testing.assert_allclose(s.x, [1.0, 0.0, 1.0], atol=1e-6)
    np.testing.assert_allclose(s.y, [1.0, 1.0], atol=1e-6)
    assert s.dual_obj == pytest.approx(1.0, abs=1e-6)


# ------------------------------------------------------------------ brute force on tiny LPs
@pytest.mark.parametrize("n,m,seed", [(4, 3, 0), (5, 4, 1), (6, 4, 2), (6, 5, 3), (7, 3, 4), (3, 2, 5)])
def test_vertex_enumeration_optimum_duality_and_complementarity(n, m, seed):
    lp = tiny.small_random(n, m, seed)
    best, xbest = vertex_enumeration(lp)
    assert np.isfinite(best)
    for pre in (dict(), dict(ruiz_iters=0, pc_alpha=0.0)):          # scaled and unscaled problem: same optimum
        s = oracle.solve(lp, eps_rel=1e-8, eps_abs=1e-8, iter_limit=400000, **pre)
        assert s.status == 0
        assert abs(s.primal_obj - best) <= 1e-6 * (1 + abs(best))
        assert abs(s.primal_obj - s.dual_obj) <= 1e-6 * (1 + abs(best))             # strong duality
        k = dense_kkt(lp, s.x, s.y)                                                 # independent numpy KKT
        assert k["rp"] <= 1e-6 and k["rd"] <= 1e-6
        assert k["pobj"] == pytest.approx(s.primal_obj, rel=1e-9, abs=1e-9)
        assert k["dobj"] == pytest.approx(s.dual_obj, rel=1e-9, abs=1e-9)
        G = lp.sense == ord("G")
        assert np.all(s.y[G] >= 0)
        assert np.abs(s.y * k["slack"]).max() <= 1e-5                               # y_i (Kx-q)_i = 0
        comp = np.where(k["lam"] > 0, k["lam"] * (s.x - np.where(np.isfinite(lp.l), lp.l, 0)),
                        k["lam"] * (s.x - np.where(np.isfinite(lp.u), lp.u, 0)))
        assert np.abs(comp).max() <= 1e-5                                           # lam_j (x_j - bound) = 0


def test_termination_measure_at_exact_optimum_and_under_perturbation():
    lp = tiny.two_var()
    k = oracle.kkt_unscaled(lp, np.array([1.0, 3.0]), np.array([1.0]))
    assert k["rel_kkt"] <= 1e-12 and k["pobj"] == -7.0 and k["dobj"] == -7.0
    # move x1 by +0.5: row -x1-x2 >= -4 violated by exactly 0.5; objective moves by -0.5
    k = oracle.kkt_unscaled(lp, np.array([1.5, 3.0]), np.array([1.0]))
    assert k["rp"] == pytest.approx(0.5, rel=1e-15) and k["rd"] == 0.0 and k["pobj"] == -7.5
    # move y by +0.25: rho = c + y = (-0.75+..): x1 has rho=-1+1.25=0.25>0 with finite lower bound -> lam, no residual
    k = oracle.kkt_unscaled(lp, np.array([1.0, 3.0]), np.array([1.25]))
    assert k["rd"] == 0.0 and k["dobj"] == pytest.approx(-4 * 1.25 + 3 * (-2 + 1.25), rel=1e-15)
    # a free variable turns the same reduced cost into a dual residual
    lp2 = tiny.free_var_lp()
    k = oracle.kkt_unscaled(lp2, np.array([1.0, 0.0, 1.0]), np.array([1.0, 0.75]))
    assert k["rd"] == pytest.approx(0.25, rel=1e-15)
    for seed in (0, 1):
        lp3 = tiny.small_random(6, 4, seed)
        s = oracle.solve(lp3, eps_rel=1e-9, eps_abs=1e-9)
        a, b = oracle.kkt_unscaled(lp3, s.x, s.y), dense_kkt(lp3, s.x, s.y)
        for key in ("rp", "rd", "pobj", "dobj"):
            assert a[key] == pytest.approx(b[key], rel=1e-12, abs=1e-14)
        # the solver's own (scaled-space) report equals the unscaled definition: identities of R1
        assert s.primal_obj == pytest.approx(a["pobj"], rel=1e-12, abs=1e-13)
        assert s.dual_obj == pytest.approx(a["dobj"], rel=1e-12, abs=1e-13)
        assert s.rel_kkt == pytest.approx(a["rel_kkt"], rel=1e-6, abs=1e-15)


# ------------------------------------------------------------------ textbook PDHG properties
def test_fejer_monotonicity_with_frozen_step():
    """With restarts off and a constant eta < 1/sigma_max(K), the PDHG-metric distance to a saddle point
    omega|x-x*|^2 + |y-y*|^2/omega + 2 eta (y-y*)'K(x-x*) never increases (Chambolle-Pock)."""
    lp = tiny.small_random(6, 4, 2)
    obj, xs, ys = highs(lp)
    k = dense_kkt(lp, xs, ys)
    assert k["rp"] < 1e-9 and k["rd"] < 1e-9 and abs(k["pobj"] - k["dobj"]) < 1e-8     # (x*, y*) is a saddle point
    K = lp.dense()
    eta = 0.9 / np.linalg.svd(K, compute_uv=False)[0]
    N = 300
    s = oracle.solve(lp, fixed_iterations=N, ruiz_iters=0, pc_alpha=0.0, frozen_eta=eta,
                     restarts_enabled=0, dump=N, trace_attempts=N)
    omega = s.omega                       # constant: no restart ever happens
    assert np.all(s.attempts["accepted"] == 1) and np.all(s.attempts["eta_used"] == eta)
    ex = s.dump_x - xs; ey = s.dump_y - ys
    d = omega * (ex ** 2).sum(1) + (ey ** 2).sum(1) / omega + 2 * eta * np.einsum("ki,ij,kj->k", ey, K, ex)
    assert np.all(d >= -1e-12)
    assert np.all(np.diff(d) <= 1e-12 * (1 + d[:-1]))
    assert d[-1] < 0.5 * d[0]


def test_average_is_eta_weighted_mean_of_accepted_iterates():
    lp = tiny.small_random(5, 4, 1)
    N = 60                                 # < check_every: no restart can clear the sums
    s = oracle.solve(lp, fixed_iterations=N, dump=N, trace_attempts=N)
    acc = s.attempts["accepted"] == 1
    w = s.attempts["eta_used"][acc]
    assert s.avg_w == pytest.approx(w.sum(), rel=1e-14)
    np.testing.assert_allclose(s.avg_x, (w[:, None] * s.dump_x[acc]).sum(0) / w.sum(), rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(s.avg_y, (w[:, None] * s.dump_y[acc]).sum(0) / w.sum(), rtol=1e-12, atol=1e-14)
    # rejected attempts leave the iterate untouched (1x1 example rejects attempt 3)
    s1 = oracle.solve(tiny.one_by_one(), fixed_iterations=4, ruiz_iters=0, pc_alpha=0.0, dump=4, trace_attempts=4)
    assert s1.attempts["accepted"][2] == 0
    assert s1.dump_x[2, 0] == s1.dump_x[1, 0] and s1.dump_y[2, 0] == s1.dump_y[1, 0]
    assert s1.accepted == 3 and s1.iterations == 4


# ------------------------------------------------------------------ R9..R11: restart rule and primal weight
@pytest.mark.parametrize("name,l,u", [("free", -np.inf, np.inf), ("bounded", 0.0, 10.0)])
def test_worked_restart_example_matches_golden(name, l, u):
    """tests/golden/restart_1x1.txt (derivation: DESIGN.md 'Worked restart example'): 13 attempts with a check after
    every one on two 1x1 LPs -- artificial, necessary and sufficient restarts, restarts to the average, a rejected
    attempt between checks, and a primal weight that moves at every restart."""
    rows = [r[1:] for r in read_golden_rows("restart_1x1.txt") if r[0] == name]
    A = [r[1:] for r in rows if r[0] == "A"]
    Cc = [r[1:] for r in rows if r[0] == "C"]
    N = len(A)
    assert N == len(Cc) == 13
    # one attempt more than the golden holds: the check at the very last attempt of a run takes no restart decision
    s = oracle.solve(tiny.one_by_one(l, u), fixed_iterations=N + 1, check_every=1, ruiz_iters=0, pc_alpha=0.0,
                     trace_attempts=N, trace_checks=N, dump=N, dump_checks=N)
    assert len(s.attempts) == N and len(s.checks) == N
    R = dict(rel=2e-9, abs=1e-12)
    x_start, y_start = 0.0, 0.0                       # the iterate attempt k starts from (R2 for k = 1)
    kinds = set()
    for i in range(N):
        k, xt, yt, eta, ebar, acc, enext = int(A[i][0]), *map(_f, A[i][1:5]), int(A[i][5]), _f(A[i][6])
        a = s.attempts[i]
        assert k == i + 1 and a["accepted"] == acc, f"attempt {k}"
        assert a["eta_used"] == pytest.approx(eta, **R) and a["eta_next"] == pytest.approx(enext, **R)
        assert a["eta_bar"] == pytest.approx(ebar, **R) if math.isfinite(ebar) else math.isinf(a["eta_bar"])
        # the iterate after attempt k (before the check): the trial point if accepted, else unchanged
        exp_x, exp_y = (xt, yt) if acc else (x_start, y_start)
        assert s.dump_x[i, 0] == pytest.approx(exp_x, **R) and s.dump_y[i, 0] == pytest.approx(exp_y, **R), f"attempt {k}"
        assert s.check_x[i, 0] == pytest.approx(exp_x, **R) and s.check_y[i, 0] == pytest.approx(exp_y, **R)
        kc, ka, cand, mu_c, mu_r, t, kind, om, xa, ya = (_f(Cc[i][1]), _f(Cc[i][2]), int(Cc[i][3]), _f(Cc[i][4]),
                                                         _f(Cc[i][5]), int(Cc[i][6]), int(Cc[i][7]), _f(Cc[i][8]),
                                                         _f(Cc[i][9]), _f(Cc[i][10]))
        c = s.checks[i]
        assert int(c["k"]) == k and c["restart_kind"] == kind, f"check {k}: kind {c['restart_kind']} != {kind}"
        if kc != ka:                                   # printed values equal = a tie decided by the last bit
            assert c["candidate"] == cand, f"check {k}"
        assert c["mu_c"] == pytest.approx(mu_c, **R) and c["mu_r"] == pytest.approx(mu_r, **R), f"check {k}"
        assert c["omega_after"] == pytest.approx(om, **R), f"check {k}"
        # where the next attempt starts: the candidate on a restart (the average if it won), else the current iterate
        if kind and c["candidate"]:
            assert s.check_avg_x[i, 0] == pytest.approx(xa, **R) and s.check_avg_y[i, 0] == pytest.approx(ya, **R)
        else:
            assert exp_x == pytest.approx(xa, **R) and exp_y == pytest.approx(ya, **R)
        x_start, y_start = xa, ya
        kinds.add((kind, c["candidate"] if kind else -1))
    assert {kd for kd, _ in kinds} == {0, 1, 2, 3}, "the example exercises no-restart and all three restart kinds"
    assert (2, 1) in kinds                             # a restart TO THE AVERAGE is part of both examples


def test_worked_restart_example_first_check_by_hand():
    """Check 1 of the 'free' example re-derived here with plain floats (DESIGN.md carries it out in words):
    z1 = (-1, 3): r_p = min(-1 - 1, 0) = -2, rho = 1 - 3 = -2 with no finite bound -> r_d = -2, pobj = -1, dobj = 3,
    KKT_1 = sqrt(4 + 4 + 16); z_r = z0 = (0, 0): r_p = -1, r_d = 1, gap 0 -> sqrt(2); t = 1 >= 0.36 -> artificial;
    Dx = 1, Dy = 3 -> omega = sqrt(1 * 3 / 1)."""
    s = oracle.solve(tiny.one_by_one(-np.inf, np.inf), fixed_iterations=3, check_every=1, ruiz_iters=0, pc_alpha=0.0,
                     trace_attempts=2, trace_checks=2)
    c1, c2 = s.checks[:2]
    assert c1["mu_c"] == pytest.approx(math.sqrt(24.0), rel=1e-15) and c1["mu_r"] == pytest.approx(math.sqrt(2.0), rel=1e-15)
    assert c1["restart_kind"] == 3 and c1["candidate"] == 0
    assert c1["omega_after"] == pytest.approx(math.sqrt(3.0), rel=1e-15)
    # check 2 evaluates the NEW restart point (-1, 3) with the NEW omega = sqrt(3): sqrt(3 * 4 + 4 / 3 + 16)
    assert c2["mu_r"] == pytest.approx(math.sqrt(12.0 + 4.0 / 3.0 + 16.0), rel=1e-15)


REPLAY_CASES = {      # name -> (LP, attempts, check_every[, weight_smoothing])
    "small_random_ce8": (lambda: tiny.small_random(6, 4, 1), 640, 8),
    "small_random_theta02": (lambda: tiny.small_random(6, 4, 1), 640, 8, 0.2),
    # the next two separate "mu_prev <- +inf on a restart" from a mu_prev that survives it (checks 4 / 4 would be kind 2)
    "small_random_c_ce8": (lambda: tiny.small_random(7, 3, 0), 400, 8),
    "small_random_ce3": (lambda: tiny.small_random(6, 4, 1), 399, 3),
    "uc0_ce16_theta08": (lambda: uc_config(0), 800, 16, 0.8),
    "small_random_b_ce5": (lambda: tiny.small_random(7, 3, 4), 640, 5),
    "free_var_ce4": (tiny.free_var_lp, 400, 4),
    "uc0": (lambda: uc_config(0), 640, 64),
    "uc0_ce16": (lambda: uc_config(0), 1600, 16),
}


def _replay_case(case):
    """R10 / R11 recomputed by helpers.restart_replay (dense numpy, closed-form geometric mean) from nothing but the
    iterates the oracle dumped at each check: candidate, restart kind, mu_c, mu_r and omega of EVERY check must be the
    oracle's.  A swapped Dy/Dx, theta vs 1 - theta, < vs <=, a stale omega in mu_r, a mu_prev that survives a restart
    or a t that does not restart at t0 each change at least one of them."""
    make, F, ce = REPLAY_CASES[case][:3]
    theta = REPLAY_CASES[case][3] if len(REPLAY_CASES[case]) > 3 else 0.5
    lp = make()
    s = oracle.solve(lp, fixed_iterations=F + 1, check_every=ce, trace_attempts=F, trace_checks=F // ce, dump_checks=F // ce,
                     weight_smoothing=theta)
    assert len(s.checks) == F // ce == len(s.check_w)
    vs, _, _ = oracle.precondition(lp)
    rep = restart_replay(lp, s, vs, theta=theta)
    seen = set()
    n_cmp = 0
    for r, c in zip(rep, s.checks):
        k = r["k"]
        if min(r["kkt_cur"], r["mu_r"]) < 1e-9:        # converged to round-off: the compared numbers are noise from here on
            break
        n_cmp += 1
        tie_c = abs(r["kkt_avg"] - r["kkt_cur"]) <= 1e-11 * r["kkt_cur"] if np.isfinite(r["kkt_avg"]) else False
        near = any(abs(r["mu_c"] - b * r["mu_r"]) <= 1e-11 * r["mu_r"] for b in (0.2, 0.8)) or \
            (np.isfinite(r["mu_prev"]) and abs(r["mu_c"] - r["mu_prev"]) <= 1e-11 * r["mu_c"])
        if not tie_c:
            assert c["candidate"] == r["candidate"], f"check at k={k}"
            assert c["mu_c"] == pytest.approx(r["mu_c"], rel=1e-9, abs=1e-13), f"k={k}"
        assert c["mu_r"] == pytest.approx(r["mu_r"], rel=1e-9, abs=1e-13), f"k={k}"
        if not (tie_c or near):
            assert c["restart_kind"] == r["kind"], f"check at k={k}: oracle {c['restart_kind']}, replay {r['kind']} ({r})"
        assert c["omega_after"] == pytest.approx(r["omega_after"], rel=1e-11), f"k={k}: Dx {r['Dx']} Dy {r['Dy']}"
        seen.add((int(c["restart_kind"]), int(c["candidate"])))
    assert n_cmp >= 10 or n_cmp == len(rep)
    # w at a check = sum of the step sizes of the attempts accepted since the last restart (R6 + 'sums <- 0' of R11)
    acc = s.attempts["accepted"] == 1
    t0 = 0
    for i, c in enumerate(s.checks):
        k = int(c["k"])
        sel = acc[t0:k]
        assert s.check_w[i] == pytest.approx(s.attempts["eta_used"][t0:k][sel].sum(), rel=1e-12), f"k={k}"
        if c["restart_kind"]:
            t0 = k
    return seen


@pytest.mark.parametrize("case", list(REPLAY_CASES))
def test_restart_decisions_and_primal_weight_recomputed_from_iterates(case):
    _replay_case(case)


def test_restart_replay_cases_cover_every_branch():
    seen = set()
    for case in REPLAY_CASES:
        seen |= _replay_case(case)
    kinds = {k for k, _ in seen}
    assert kinds == {0, 1, 2, 3}, seen
    assert {c for k, c in seen if k} == {0, 1}, "restarts to the current iterate and to the average both occur"


def test_restart_and_primal_weight_invariants():
    lp = uc_config(0)
    s = oracle.solve(lp, fixed_iterations=640)
    assert len(s.checks) == 10 and s.checks["k"].tolist() == [64 * i for i in range(1, 11)]
    assert s.checks["restart_kind"][0] == 3            # t = k at the first check: artificial restart fires
    assert np.all(np.isfinite(s.checks["omega_after"])) and np.all(s.checks["omega_after"] > 0)
    assert s.restarts == int((s.checks["restart_kind"][:-1] > 0).sum()) + int(s.checks["restart_kind"][-1] > 0)
    # no restart when disabled; omega then never changes
    s2 = oracle.solve(lp, fixed_iterations=256, restarts_enabled=0)
    assert s2.restarts == 0 and np.all(s2.checks["restart_kind"] == 0)
    assert np.all(s2.checks["omega_after"] == s2.checks["omega_after"][0])
    # after a restart at k=64 the weighted sums restart: with F=64+1 the average holds one iterate
    s3 = oracle.solve(lp, fixed_iterations=65, trace_attempts=65, dump=65)
    assert s3.avg_w == pytest.approx(s3.attempts["eta_used"][64], rel=1e-15)
    np.testing.assert_allclose(s3.avg_x, s3.dump_x[64], rtol=1e-13, atol=1e-300)
    # box-only LP: y-space is empty so Delta_y = 0 <= 1e-10 and omega must stay at its initial value 1
    s4 = oracle.solve(tiny.box_only(5, 2), fixed_iterations=200)
    assert np.all(s4.checks["omega_after"] == 1.0)


def test_status_codes_and_iteration_accounting():
    lp = uc_config(0)
    s = oracle.solve(lp, iter_limit=100)
    assert s.status == 1 and s.iterations == 100 and len(s.checks) == 2           # checks at 64 and at the cap
    s = oracle.solve(lp, fixed_iterations=200, trace_attempts=200)
    assert s.iterations == 200 and len(s.attempts) == 200 and s.accepted == int(s.attempts["accepted"].sum())
    assert len(s.checks) == 3 and s.returned_average == 0


# ------------------------------------------------------------------ R12 with eps_abs != eps_rel; which point a capped run returns
def _dense_terms(lp, s, i):
    """dense_kkt of the current iterate and of the average that check i of an oracle run saw (unscaled from its dumps)."""
    cur = dense_kkt(lp, s.check_x[i] / s.Dc, s.check_y[i] / s.Dr)
    avg = dense_kkt(lp, s.check_avg_x[i] / s.Dc, s.check_avg_y[i] / s.Dr)
    return cur, avg


def _passes(lp, k, ea, er):
    """R12 / SURVEY O5 written out: ||r_p|| <= ea + er ||q||, ||r_d|| <= ea + er ||c||, |gap| <= ea + er (|p| + |d|)."""
    return (k["rp"] <= ea + er * np.linalg.norm(lp.b) and k["rd"] <= ea + er * np.linalg.norm(lp.c) and
            abs(k["pobj"] - k["dobj"]) <= ea + er * (abs(k["pobj"]) + abs(k["dobj"])))


@pytest.mark.parametrize("name", ["small_random", "uc0"])
@pytest.mark.parametrize("ea,er", [(1e-3, 1e-9), (1e-9, 1e-3), (1e-5, 1e-4)])
def test_termination_with_separate_absolute_and_relative_tolerances(name, ea, er):
    """PAPER.md l.66 sets an ABSOLUTE feasibility tolerance (1e-5) next to the relative 1e-4 of l.91, so eps_abs and eps_rel
    differ in the paper's own runs.  From the iterates the oracle dumped at every check, dense numpy algebra decides where
    the run had to stop: at the FIRST check whose average or current iterate passes R12 with (ea, er) in their own places.
    The oracle with the two swapped (or one used for both) stops at a different check on these LPs -- asserted below, so
    the case really separates them."""
    lp = tiny.small_random(6, 4, 1) if name == "small_random" else uc_config(0)
    s = oracle.solve(lp, eps_abs=ea, eps_rel=er, iter_limit=400000, dump_checks=8192, trace_checks=8192)
    assert s.status == 0 and len(s.check_x) == len(s.checks) < 8192
    last = len(s.checks) - 1
    for i in range(last + 1):
        cur, avg = _dense_terms(lp, s, i)
        ok_avg, ok_cur = _passes(lp, avg, ea, er), _passes(lp, cur, ea, er)
        if i < last:
            # a borderline value (within rounding of the threshold) would make this comparison of two different
            # summation orders meaningless; none occurs on these LPs
            assert not ok_avg and not ok_cur, f"check {i} already passes but the oracle went on"
        else:
            assert ok_avg or ok_cur, "oracle stopped at a check that does not pass"
            assert s.returned_average == (1 if ok_avg else 0)           # the average is tried first (R12)
    if ea != er and not (ea, er) == (1e-5, 1e-4):
        swapped = oracle.solve(lp, eps_abs=er, eps_rel=ea, iter_limit=400000)
        assert swapped.iterations != s.iterations                        # the pair is not symmetric on this LP


@pytest.mark.parametrize("name,limit", [("uc0", 100), ("uc0", 640), ("small_random", 64), ("small_random", 192)])
def test_a_run_that_hits_its_iteration_limit_returns_the_better_of_current_and_average(name, limit):
    """R12 / SURVEY O5: on a non-OPTIMAL exit the point handed back is whichever of the current iterate and the average has
    the smaller relative KKT error at the last check (ties: the current one).  Decided here by dense numpy algebra on the
    dumped iterates, with the relative KKT error written out from its definition (R9)."""
    lp = tiny.small_random(6, 4, 1) if name == "small_random" else uc_config(0)
    s = oracle.solve(lp, iter_limit=limit, eps_abs=0.0, eps_rel=0.0, dump_checks=64, trace_checks=64)
    assert s.status == 1 and s.iterations == limit and int(s.checks["k"][-1]) == limit
    cur, avg = _dense_terms(lp, s, len(s.checks) - 1)

    def rel(k):
        return max(k["rp"] / (1 + np.linalg.norm(lp.b)), k["rd"] / (1 + np.linalg.norm(lp.c)),
                   abs(k["pobj"] - k["dobj"]) / (1 + abs(k["pobj"]) + abs(k["dobj"])))
    rc, ra = rel(cur), rel(avg)
    assert abs(rc - ra) > 1e-9 * max(rc, ra)                             # not a tie: the choice is decided
    want_avg = ra < rc and s.check_w[-1] > 0.0
    assert s.returned_average == int(want_avg)
    i = len(s.checks) - 1
    xs, ys = (s.check_avg_x[i], s.check_avg_y[i]) if want_avg else (s.check_x[i], s.check_y[i])
    np.testing.assert_array_equal(s.x, xs / s.Dc)
    np.testing.assert_array_equal(s.y, ys / s.Dr)
    assert s.rel_kkt == pytest.approx(min(rc, ra) if s.check_w[-1] > 0.0 else rc, rel=1e-6)


# ------------------------------------------------------------------ R2b: a run that starts from a supplied step size and primal weight
def test_supplied_step_size_and_primal_weight_are_the_ones_the_first_attempt_and_check_use():
    """R2b.  LP: min x s.t. x >= 1, x free; K = [1], c = q = 1, no preconditioning,
    x0 = y0 = 0, a check after every attempt, eta0 = 0.5, omega0 = 4 (R2's own values would be 1 and 1).  By hand:
      attempt 1: tau = eta/omega = 1/8, x' = 0 - (1 - 0)/8 = -1/8, xbar = -1/4; sigma = eta*omega = 2, y' = max(0, 0 + 2 (1 + 1/4)) = 5/2
                 dx2 = 1/64, dy2 = 25/4, |dy K dx| = 5/16, eta_bar = (4/64 + 25/16) / (2 * 5/16) = 2.6 >= 0.5: accepted
      check 1 (weight 4): current point: r_p = min(-1/8 - 1, 0) = -9/8, r_d = 1 - 5/2 = -3/2 (x free), gap = -1/8 - 5/2 = -21/8
                 mu_c = sqrt(16 * 81/64 + (9/4)/16 + 441/64) = sqrt(27.28125)
                 restart point (0, 0): r_p = -1, r_d = 1, gap = 0: mu_r = sqrt(16 + 1/16) = sqrt(16.0625)
    Every value is exact in binary, so the comparisons are exact up to the square roots."""
    from workloads.lp import from_dense
    lp = from_dense([[1.0]], ["G"], [1.0], [1.0], [-np.inf], [np.inf], name="free_1x1")
    kw = dict(ruiz_iters=0, pc_alpha=0.0, check_every=1, fixed_iterations=1, trace_attempts=1, trace_checks=1)
    s = oracle.solve(lp, eta0=0.5, omega0=4.0, **kw)
    a = s.attempts[0]
    assert (a["eta_used"], a["dx2"], a["dy2"], a["inter"], a["eta_bar"], a["accepted"]) == (0.5, 1 / 64, 25 / 4, 5 / 16, 2.6, 1)
    assert (s.x[0], s.y[0]) == (-0.125, 2.5)
    kw2 = dict(kw, fixed_iterations=2, trace_attempts=2, trace_checks=2)         # the restart test runs only before the last attempt
    c = oracle.solve(lp, eta0=0.5, omega0=4.0, **kw2).checks[0]
    assert c["k"] == 1
    assert c["mu_c"] == pytest.approx(np.sqrt(27.28125), rel=1e-15) and c["mu_r"] == pytest.approx(np.sqrt(16.0625), rel=1e-15)
    # one at a time: the other one keeps R2's value (1 and 1 on this LP)
    s = oracle.solve(lp, eta0=0.5, **kw)
    assert (s.attempts[0]["eta_used"], s.x[0], s.y[0]) == (0.5, -0.5, 1.0)                  # tau = sigma = 1/2: x' = -1/2, y' = (1 + 1)/2
    s = oracle.solve(lp, omega0=4.0, **kw)
    assert (s.attempts[0]["eta_used"], s.x[0], s.y[0]) == (1.0, -0.25, 6.0)                 # tau = 1/4, sigma = 4: y' = 4 (1 + 1/2)
    # 0 = not supplied: the run is R2's, bit for bit
    d = oracle.solve(uc_config(0), fixed_iterations=130, trace_attempts=130)
    z = oracle.solve(uc_config(0), fixed_iterations=130, trace_attempts=130, eta0=0.0, omega0=0.0)
    np.testing.assert_array_equal(d.x, z.x); np.testing.assert_array_equal(d.attempts["eta_used"], z.attempts["eta_used"])
    # and a run continued from the state of another ends where a longer run of the same attempts would not be reproduced
    # exactly (k restarts from 1), but its first step size IS the supplied one
    w = oracle.solve(uc_config(0), x0=d.x, y0=d.y, eta0=d.eta, omega0=d.omega, fixed_iterations=1, trace_attempts=1)
    assert w.attempts["eta_used"][0] == d.eta


# ------------------------------------------------------------------ library cross-check on the UC LP
def test_uc_config0_converges_to_highs_objective():
    lp = uc_config(0)
    obj, xh, yh = highs(lp)
    s = oracle.solve(lp)
    assert s.status == 0 and s.rel_kkt <= 1e-4
    assert abs(s.primal_obj - obj) <= 1e-3 * (1 + abs(obj))
    k = oracle.kkt_unscaled(lp, s.x, s.y)
    assert k["rel_kkt"] == pytest.approx(s.rel_kkt, rel=1e-6)
    # HiGHS's own primal-dual pair is optimal under the oracle's KKT definition (sign convention pin)
    kh = oracle.kkt_unscaled(lp, xh, yh)
    assert kh["rel_kkt"] <= 1e-7
    # tighter tolerance moves the objective closer
    s2 = oracle.solve(lp, eps_rel=1e-7, eps_abs=1e-7, iter_limit=400000)
    assert s2.status == 0 and abs(s2.primal_obj - obj) <= 1e-5 * (1 + abs(obj))


def test_fixed_commitment_objective_not_below_relaxed():
    """north_star: 'commitment relaxed to [0,1] or fixed' -- fixing u to a 0/1 pattern (l_j = u_j)."""
    lp = uc_config(0)
    G, T, V, oU = lp.meta["G"], lp.meta["T"], lp.meta["V"], lp.meta["offsets"]["u"]
    relaxed = oracle.solve(lp)
    pattern = (relaxed.x.reshape(T, V)[:, oU:oU + G].T > 0.5).astype(float)
    lpf = fix_commitment(lp, pattern)
    obj, _, _ = highs(lpf)                       # feasible for this pattern (HiGHS asserts optimal)
    fixed = oracle.solve(lpf)
    assert fixed.status == 0
    assert fixed.primal_obj >= relaxed.primal_obj * (1 - 1e-3)
    assert abs(fixed.primal_obj - obj) <= 1e-3 * (1 + abs(obj))
    np.testing.assert_allclose(fixed.x.reshape(T, V)[:, oU:oU + G].T, pattern, rtol=0, atol=1e-14)   # clamp keeps l = u


def test_warm_start_from_solution_terminates_at_first_check():
    lp = tiny.small_random(6, 4, 0)
    s = oracle.solve(lp, eps_rel=1e-9, eps_abs=1e-9)
    s2 = oracle.solve(lp, x0=s.x, y0=s.y, eps_rel=1e-6, eps_abs=1e-6)
    assert s2.status == 0 and s2.iterations == 64
