"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI (ctypes binding), against the CPU
oracle on the same seeded inputs.  Bars (BASELINE.json north_star): after a fixed 200 attempts the
iterates agree within 1e-10 relative L2 (x and y separately) with identical accept / restart traces;
at convergence (relative KKT <= 1e-4) objectives agree within 1e-5 relative.  Integer / index work
(layout round trip, K' == CSC(K)) is compared bit-exactly."""
import json
import os

import numpy as np
import pytest

import oracle
import paper_2607_03627_b200 as P
from workloads import tiny, uc_config, random_lp, fix_commitment
from workloads.lp import LP, from_dense

from helpers import rel_l2, highs, GOLDEN

pytestmark = pytest.mark.gpu

TOL_ITER = 1e-10     # north_star: iterates after 200 fixed attempts, relative L2
TOL_OBJ = 1e-5       # north_star: objectives at convergence, relative


def ragged_lp(seed=5, n=3000, m=2500):
    """Random LP with empty rows, empty columns, a few rows far longer than the sliced-ELL threshold
    and a ragged tail (sizes not multiples of 32)."""
    rng = np.random.default_rng(seed)
    n, m = n + 7, m + 13
    lens = rng.integers(0, 9, m)
    lens[rng.integers(0, m, 5)] = rng.integers(40, 400, 5)          # long tail rows
    lens[:3] = 0
    rows, cols = [], []
    for i, k in enumerate(lens):
        c = rng.choice(n - 11, size=int(k), replace=False)           # last 11 columns stay empty
        rows += [i] * int(k); cols += c.tolist()
    vals = rng.standard_normal(len(rows)) * rng.choice([0.01, 1.0, 50.0], len(rows))
    l = -rng.uniform(0, 5, n); u = rng.uniform(0, 5, n)
    l[rng.integers(0, n, 40)] = -np.inf; u[rng.integers(0, n, 40)] = np.inf
    x0 = np.clip(rng.standard_normal(n), np.maximum(l, -3), np.minimum(u, 3))
    from workloads.lp import from_coo
    sense = np.where(rng.uniform(size=m) < 0.4, ord("E"), ord("G")).astype(np.uint8)
    lp = from_coo(m, n, rows, cols, vals, sense, np.zeros(m), rng.standard_normal(n), l, u, name="ragged")
    lp.b = lp.to_scipy() @ x0 - np.where(sense == ord("G"), rng.uniform(0, 1, m), 0.0)
    return lp


def shuffled_in_rows(lp, seed):
    """The same LP with the entries of every row in a random order (include/uc_pdhg.h: "order inside a row is free").
    Built here on the raw CSR arrays: workloads.lp.from_coo would sort the columns again.  The sum of a row follows the
    caller's storage order on both sides, so the oracle is given the shuffled LP too and parity stays bit-level."""
    import copy
    rng = np.random.default_rng(seed)
    q = copy.copy(lp)
    q.col_idx = lp.col_idx.copy(); q.val = lp.val.copy()
    for i in range(lp.m):
        a, b = int(lp.row_ptr[i]), int(lp.row_ptr[i + 1])
        if b - a > 1:
            p = a + rng.permutation(b - a)
            q.col_idx[a:b] = lp.col_idx[p]; q.val[a:b] = lp.val[p]
    assert any(np.any(np.diff(q.col_idx[int(q.row_ptr[i]):int(q.row_ptr[i + 1])]) < 0) for i in range(min(lp.m, 200)))
    q.name = lp.name + "_shuffled"
    return q


CASES = {
    "one_by_one": tiny.one_by_one,
    "two_var": tiny.two_var,
    "box_only": lambda: tiny.box_only(),
    "box_rows": lambda: tiny.box_only(with_rows=3),
    "free_var": tiny.free_var_lp,
    "small_random": lambda: tiny.small_random(6, 4, 1),
    "dispatch": lambda: tiny.economic_dispatch()[0],
    "ragged": ragged_lp,
    "uc0": lambda: uc_config(0),
    "uc1": lambda: uc_config(1),
    "random_2e4": lambda: random_lp(20_000, 21),
    "tuned_presolve": lambda: uc_config("tuned_presolve"),        # the shape PAPER.md l.232 / Table VI is about
    "uc1_shuffled": lambda: shuffled_in_rows(uc_config(1), 7),
    "ragged_shuffled": lambda: shuffled_in_rows(ragged_lp(), 8),
}
_lp_cache = {}


def get_lp(name):
    if name not in _lp_cache:
        _lp_cache[name] = CASES[name]()
    return _lp_cache[name]


def assert_trajectory_parity(lp, F=200, **opts):
    so = oracle.solve(lp, fixed_iterations=F, trace_attempts=F, trace_checks=64)
    with P.UcLp(lp, **opts) as h:
        sg = h.solve(fixed_iterations=F, trace_attempts=F, trace_checks=64)
    assert sg.status == P.ITERATION_LIMIT and sg.iterations == F == so.iterations
    np.testing.assert_array_equal(sg.attempts["accepted"], so.attempts["accepted"])
    np.testing.assert_array_equal(sg.checks["k"], so.checks["k"])
    np.testing.assert_array_equal(sg.checks["restart_kind"], so.checks["restart_kind"])
    np.testing.assert_array_equal(sg.checks["candidate"], so.checks["candidate"])
    assert rel_l2(sg.x, so.x) <= TOL_ITER, "x after %d attempts" % F
    if lp.m:
        assert rel_l2(sg.y, so.y) <= TOL_ITER, "y after %d attempts" % F
    np.testing.assert_allclose(sg.attempts["eta_used"], so.attempts["eta_used"], rtol=1e-9)
    assert sg.accepted == so.accepted and sg.restarts == so.restarts
    assert sg.omega == pytest.approx(so.omega, rel=1e-9) and sg.eta == pytest.approx(so.eta, rel=1e-9)
    assert sg.primal_obj == pytest.approx(so.primal_obj, rel=1e-9, abs=1e-9)
    assert sg.rel_kkt == pytest.approx(so.rel_kkt, rel=1e-6, abs=1e-12)
    return sg, so


# ------------------------------------------------------------------ A1: ingest on the device (integer work: bit-exact)
def banded_and_wide_lp(n=60_000, m=45_000, seed=4):
    """Narrow-band rows (16-bit offsets apply) mixed with rows that reach across all columns (32-bit slices)."""
    from workloads.lp import from_coo
    rng = np.random.default_rng(seed)
    rows, cols = [], []
    for i in range(m):
        k = int(rng.integers(1, 6))
        if i % 97 == 0:
            c = rng.choice(n, size=k, replace=False)
        else:
            base = int(i * (n - 300) / m)
            c = base + rng.choice(300, size=k, replace=False)
        rows += [i] * k; cols += c.tolist()
    vals = rng.standard_normal(len(rows))
    return from_coo(m, n, rows, cols, vals, np.full(m, ord("G"), np.uint8), -np.ones(m), rng.standard_normal(n), -np.ones(n), np.ones(n), name="banded")


INGEST_CASES = dict(CASES, banded=banded_and_wide_lp, random_3e5=lambda: random_lp(300_000, 22), uc2=lambda: uc_config(2))


@pytest.mark.parametrize("name", list(INGEST_CASES))
@pytest.mark.parametrize("window,thr,compress", [(4096, 32, 1), (64, 3, 1), (4096, 1000, 0)])
def test_device_ingest_builds_the_host_layouts_bit_for_bit(name, window, thr, compress):
    """uc_lp_create with host_ingest = 0 (kernels: stable radix sorts, scans, per-row fills) must leave on the device
    exactly what the host builders -- verified against the caller's CSR by uc_host_layout_selftest -- produce:
    permutations, slice pointers, 32-bit indices / 16-bit offsets, values, long rows, schedules.  No preconditioning,
    so that the values can be compared too."""
    if name not in INGEST_CASES:
        pytest.skip()
    lp = INGEST_CASES[name]() if name not in CASES else get_lp(name)
    with P.UcLp(lp, sell_window=window, long_row_threshold=thr, index_compression=compress, ruiz_iters=0, pc_alpha=0.0, host_ingest=0) as h:
        h.compare_layout(lp)
    with P.UcLp(lp, sell_window=window, long_row_threshold=thr, index_compression=compress, ruiz_iters=0, pc_alpha=0.0, host_ingest=1) as h:
        h.compare_layout(lp)                                  # the checker agrees with itself through the upload path


def test_device_and_host_ingest_give_identical_solves():
    lp = get_lp("uc1")
    with P.UcLp(lp, host_ingest=0) as a, P.UcLp(lp, host_ingest=1) as b:
        sa = a.solve(fixed_iterations=200, trace_attempts=200); sb = b.solve(fixed_iterations=200, trace_attempts=200)
    np.testing.assert_array_equal(sa.x, sb.x); np.testing.assert_array_equal(sa.y, sb.y)
    np.testing.assert_array_equal(sa.attempts["eta_used"], sb.attempts["eta_used"])


def test_paper_scale_config3_device_ingest_matches_host_layouts():
    lp = uc_config(3)
    with P.UcLp(lp, ruiz_iters=0, pc_alpha=0.0) as h:
        h.compare_layout(lp)


# ------------------------------------------------------------------ R1: preconditioner + layouts
@pytest.mark.parametrize("name", ["two_var", "small_random", "ragged", "uc0", "uc1", "random_2e4"])
def test_preconditioner_matches_oracle(name):
    lp = get_lp(name)
    vs, Dr, Dc = oracle.precondition(lp)
    with P.UcLp(lp, keep_source_map=1) as h:
        gDr, gDc = h.scaling()
        v_k, v_kt = h.scaled_values(False), h.scaled_values(True)
    np.testing.assert_allclose(gDr, Dr, rtol=1e-14)
    np.testing.assert_allclose(gDc, Dc, rtol=1e-14)
    np.testing.assert_allclose(v_k, vs, rtol=1e-14)
    np.testing.assert_array_equal(v_k, v_kt)          # K' is the CSC of K, bit for bit, after 11 scaling passes


@pytest.mark.parametrize("alpha,ruiz", [(0.0, 10), (1.0, 0), (0.0, 0)])
def test_preconditioner_options(alpha, ruiz):
    lp = get_lp("uc0")
    vs, Dr, Dc = oracle.precondition(lp, ruiz_iters=ruiz, pc_alpha=alpha)
    with P.UcLp(lp, keep_source_map=1, ruiz_iters=ruiz, pc_alpha=alpha) as h:
        gDr, gDc = h.scaling()
        np.testing.assert_allclose(h.scaled_values(False), vs, rtol=1e-14)
    np.testing.assert_allclose(gDr, Dr, rtol=1e-14)
    np.testing.assert_allclose(gDc, Dc, rtol=1e-14)


@pytest.mark.parametrize("alpha,ruiz", [(0.5, 10), (1.5, 2)])
def test_pock_chambolle_general_exponent(alpha, ruiz):
    """alpha != 1 takes the `pow` branch of k_row_stat (mode 2).  CUDA's pow is 2-ulp accurate where the oracle's libm pow
    is correctly rounded, so the bar is not bit equality: a sum of positive terms keeps the relative error of its terms
    (<= 2 ulp = 4.4e-16), the square root halves it and the division by r_i * s_j adds both: < 1e-15 per value; 1e-13
    leaves room for the ordering of the sums.  The two layouts must still agree bit for bit (same r_i * s_j in both).
    The trajectories are then NOT bit-identical (the scaled problems differ in the last bits), so the two solves stop at
    different points of the same 1e-4 relative KKT ball: their objectives agree to that accuracy, not to 1e-5."""
    lp = get_lp("uc0")
    vs, Dr, Dc = oracle.precondition(lp, ruiz_iters=ruiz, pc_alpha=alpha)
    with P.UcLp(lp, keep_source_map=1, ruiz_iters=ruiz, pc_alpha=alpha) as h:
        gDr, gDc = h.scaling()
        v_k, v_kt = h.scaled_values(False), h.scaled_values(True)
        sg = h.solve()
    np.testing.assert_allclose(v_k, vs, rtol=1e-13)
    np.testing.assert_allclose(gDr, Dr, rtol=1e-13)
    np.testing.assert_allclose(gDc, Dc, rtol=1e-13)
    np.testing.assert_array_equal(v_k, v_kt)
    so = oracle.solve(lp, ruiz_iters=ruiz, pc_alpha=alpha)
    assert sg.status == P.OPTIMAL and so.status == 0 and sg.rel_kkt <= 1e-4
    assert abs(sg.primal_obj - so.primal_obj) <= 5e-4 * abs(so.primal_obj)


@pytest.mark.parametrize("name", ["small_random", "ragged", "uc1"])
def test_spmv_pair_matches_oracle_and_is_adjoint(name):
    lp = get_lp(name)
    rng = np.random.default_rng(3)
    x = rng.standard_normal(lp.n); y = rng.standard_normal(lp.m)
    vs, _, _ = oracle.precondition(lp)
    with P.UcLp(lp) as h:
        kx = h.spmv(x, transpose=False)
        kty = h.spmv(y, transpose=True)
    ox, oty = oracle.spmv(lp, x, val=vs), oracle.spmv_t(lp, y, val=vs)
    assert rel_l2(kx, ox) <= 1e-13 and rel_l2(kty, oty) <= 1e-13
    assert abs(y @ kx - kty @ x) <= 1e-12 * (np.abs(y) @ np.abs(kx) + 1.0)       # adjoint identity


# ------------------------------------------------------------------ A5..A9 at kernel level: ONE attempt, restated in numpy
@pytest.mark.parametrize("name", ["small_random", "ragged", "uc0", "uc1", "random_2e4"])
def test_one_attempt_of_the_attempt_kernels_matches_a_numpy_restatement(name):
    """k_primal + k_dual once, from a random warm start, against R2..R5 written out with scipy on the oracle's scaled
    matrix: g = K~'y~, x' = clamp(x~ - tau (c~ - g)), xbar = 2x' - x~, y' = proj(y~ + sigma (q~ - K~ xbar)) and the three
    reductions of the step rule.  This is the kernel-level tier for the pipelines of uc_attempt.cuh (uc_lp_spmv runs the
    check kernels' traversal, not these)."""
    import scipy.sparse as sp
    lp = get_lp(name)
    rng = np.random.default_rng(11)
    x0 = rng.standard_normal(lp.n); y0 = rng.standard_normal(lp.m)
    vs, Dr, Dc = oracle.precondition(lp)
    K = sp.csr_matrix((vs, lp.col_idx, lp.row_ptr), shape=(lp.m, lp.n))
    isG = np.asarray(lp.sense) == ord("G")
    c, q = lp.c / Dc, lp.b / Dr
    l = np.where(lp.l <= -1e20, -np.inf, lp.l * Dc); u = np.where(lp.u >= 1e20, np.inf, lp.u * Dc)
    x = np.clip(x0 * Dc, l, u); y = y0 * Dr; y[isG] = np.maximum(y[isG], 0.0)                      # R2
    eta = 1.0 / np.abs(vs).max() if lp.nnz else 1.0
    nc, nq = np.linalg.norm(c), np.linalg.norm(q)
    omega = nc / nq if nc > 1e-10 and nq > 1e-10 else 1.0
    xn = np.clip(x - (eta / omega) * (c - K.T @ y), l, u); xbar = 2.0 * xn - x                       # R3
    yn = y + eta * omega * (q - K @ xbar); yn[isG] = np.maximum(yn[isG], 0.0)                       # R4
    dx, dy = xn - x, yn - y
    dx2, dy2, inter = float(dx @ dx), float(dy @ dy), abs(float(dy @ (K @ dx)))                     # R5
    with P.UcLp(lp) as h:
        s = h.solve(x0=x0, y0=y0, fixed_iterations=1, trace_attempts=1)
    a = s.attempts[0]
    assert a["eta_used"] == pytest.approx(eta, rel=1e-14)
    assert a["dx2"] == pytest.approx(dx2, rel=1e-12) and a["dy2"] == pytest.approx(dy2, rel=1e-12)
    assert a["inter"] == pytest.approx(inter, rel=1e-9, abs=1e-12 * (dx2 + dy2))
    N = omega * dx2 + dy2 / omega
    assert bool(a["accepted"]) == (eta <= (N / (2 * inter) if inter > 0 else np.inf))
    ex, ey = (xn, yn) if a["accepted"] else (x, y)
    assert rel_l2(s.x, ex / Dc) <= 1e-12
    if lp.m:
        assert rel_l2(s.y, ey / Dr) <= 1e-12


# ------------------------------------------------------------------ R2..R11: 200-attempt trajectory
@pytest.mark.parametrize("name", list(CASES))
def test_trajectory_parity_200_attempts(name):
    assert_trajectory_parity(get_lp(name), 200)


def test_trajectory_parity_uc2_medium():
    assert_trajectory_parity(uc_config(2), 200)


@pytest.mark.parametrize("name", ["uc1_shuffled", "ragged_shuffled"])
def test_rows_stored_in_any_column_order_pass_the_layout_checks(name):
    """Unsorted rows through the host self-check (entries kept in the caller's order) and the device-vs-host ingest
    comparison; their 200-attempt parity runs with the other CASES."""
    lp = get_lp(name)
    from paper_2607_03627_b200.binding import host_layout_selftest
    host_layout_selftest(lp)
    host_layout_selftest(lp, sell_window=64, long_row_threshold=3)
    with P.UcLp(lp, ruiz_iters=0, pc_alpha=0.0) as h:
        h.compare_layout(lp)
    with P.UcLp(lp, sell_window=64, long_row_threshold=3, ruiz_iters=0, pc_alpha=0.0) as h:
        h.compare_layout(lp)


@pytest.mark.parametrize("big", [1e20, 1e30])
def test_finite_sentinel_bounds_are_absent_bounds_on_both_sides(big):
    """R13: |bound| >= 1e20 means "no bound".  uc_config(0) with every infinite bound written as +-1e20
    / +-1e30 must give, on each side, the very bits of the +-inf run -- and the GPU run the oracle's trajectory."""
    import copy
    lp = get_lp("uc0")
    q = copy.copy(lp)
    q.l = np.where(np.isneginf(lp.l), -big, lp.l); q.u = np.where(np.isposinf(lp.u), big, lp.u)
    assert (np.isinf(lp.l).sum() + np.isinf(lp.u).sum()) > 0 and not np.isinf(q.l).any() and not np.isinf(q.u).any()
    so_inf = oracle.solve(lp, fixed_iterations=200); so_big = oracle.solve(q, fixed_iterations=200)
    np.testing.assert_array_equal(so_big.x, so_inf.x); np.testing.assert_array_equal(so_big.y, so_inf.y)
    assert (so_big.primal_obj, so_big.dual_obj, so_big.rel_kkt) == (so_inf.primal_obj, so_inf.dual_obj, so_inf.rel_kkt)
    with P.UcLp(lp) as a, P.UcLp(q) as b:
        sa = a.solve(fixed_iterations=200, trace_attempts=200); sb = b.solve(fixed_iterations=200, trace_attempts=200)
    np.testing.assert_array_equal(sb.x, sa.x); np.testing.assert_array_equal(sb.y, sa.y)
    np.testing.assert_array_equal(sb.attempts["eta_used"], sa.attempts["eta_used"])
    assert (sb.primal_obj, sb.dual_obj, sb.rel_kkt) == (sa.primal_obj, sa.dual_obj, sa.rel_kkt)
    assert_trajectory_parity(q, 200)


@pytest.mark.parametrize("what,k_fail", [("matrix", 1), ("cost", 64), ("rhs_tiny_matrix", 64)])
def test_overflowing_input_ends_in_numerical_error_at_the_oracles_attempt(what, k_fail):
    """R12: a non-finite step size stops the run at that attempt (the step rule in the dual kernel), a non-finite KKT term at
    the next check.  Without preconditioning, entries of 1e200 overflow dx'K'dy in the first attempt; a cost of 1e308
    or a right-hand side of 1e200 over a 1e-200 matrix overflow the objectives at the first check."""
    import copy
    q = copy.copy(get_lp("small_random"))
    if what == "matrix":
        q.val = q.val * 1e200
    elif what == "cost":
        q.c = q.c / np.abs(q.c).max() * 1e308
    else:
        q.val = q.val * 1e-200; q.b = q.b * 1e200
    so = oracle.solve(q, ruiz_iters=0, pc_alpha=0.0, iter_limit=1000)
    assert so.status == 4 and so.iterations == k_fail
    with P.UcLp(q, ruiz_iters=0, pc_alpha=0.0) as h:
        sg = h.solve(iter_limit=1000)
        assert sg.status == P.NUMERICAL_ERROR and sg.iterations == so.iterations
        assert h.solve(iter_limit=1000).status == P.NUMERICAL_ERROR       # and the handle survives it


@pytest.mark.parametrize("window,thr", [(32, 4), (64, 1), (100000, 1000)])
def test_trajectory_parity_is_layout_independent(window, thr):
    """Other slicing windows / long-row thresholds (all rows long, no row long) give the same iterates."""
    assert_trajectory_parity(get_lp("ragged"), 130, sell_window=window, long_row_threshold=thr)


@pytest.mark.parametrize("name", ["uc1", "ragged", "random_2e4"])
def test_index_compression_is_bit_identical(name):
    """SURVEY.md 8(f) NEXT-4, 16-bit column offsets inside a slice: integer work, so the iterates with and without it are
    the same bits (and both match the oracle through test_trajectory_parity_200_attempts)."""
    lp = get_lp(name)
    with P.UcLp(lp, index_compression=1) as h:
        a = h.solve(fixed_iterations=300)
        ia = h.info()
    with P.UcLp(lp, index_compression=0) as h:
        b = h.solve(fixed_iterations=300)
        ib = h.info()
    np.testing.assert_array_equal(a.x, b.x); np.testing.assert_array_equal(a.y, b.y)
    assert ib.k_narrow_slots == ib.kt_narrow_slots == 0
    assert ib.bytes_per_attempt - ia.bytes_per_attempt == 2 * (ia.k_narrow_slots + ia.kt_narrow_slots)
    if name == "uc1":       # period-local structure: every slice of K is narrow; in K' the reserve columns reach the long
        assert ia.k_narrow_slots == ia.k_sell_slots         # reserve rows, which sit at the end of the permuted row space
        assert 0.95 * ia.kt_sell_slots <= ia.kt_narrow_slots <= ia.kt_sell_slots


def test_index_compression_mixed_narrow_and_wide_slices():
    from test_layout_cpu import banded_and_wide_lp
    lp = banded_and_wide_lp()
    so = oracle.solve(lp, fixed_iterations=130)
    with P.UcLp(lp) as h:
        sg = h.solve(fixed_iterations=130)
        i = h.info()
    assert 0 < i.k_narrow_slots < i.k_sell_slots
    assert rel_l2(sg.x, so.x) <= TOL_ITER and rel_l2(sg.y, so.y) <= TOL_ITER


def test_trajectory_parity_other_check_period_and_tail():
    lp = get_lp("uc0")
    for F, ce in ((37, 10), (64, 64), (65, 64), (1, 64)):
        so = oracle.solve(lp, fixed_iterations=F, check_every=ce, trace_checks=64)
        with P.UcLp(lp) as h:
            sg = h.solve(fixed_iterations=F, check_every=ce, trace_checks=64)
        assert rel_l2(sg.x, so.x) <= TOL_ITER and rel_l2(sg.y, so.y) <= TOL_ITER
        np.testing.assert_array_equal(sg.checks["restart_kind"], so.checks["restart_kind"])
        assert sg.iterations == F


def test_warm_start_parity():
    lp = get_lp("uc0")
    rng = np.random.default_rng(9)
    x0 = rng.uniform(-1, 2, lp.n); y0 = rng.standard_normal(lp.m)
    so = oracle.solve(lp, x0=x0, y0=y0, fixed_iterations=100)
    with P.UcLp(lp) as h:
        sg = h.solve(x0=x0, y0=y0, fixed_iterations=100)
    assert rel_l2(sg.x, so.x) <= TOL_ITER and rel_l2(sg.y, so.y) <= TOL_ITER


# ------------------------------------------------------------------ convergence parity
@pytest.mark.parametrize("name", ["two_var", "free_var", "small_random", "dispatch", "uc0"])
def test_convergence_parity_live(name):
    lp = get_lp(name)
    so = oracle.solve(lp)
    with P.UcLp(lp) as h:
        sg = h.solve()
    assert sg.status == P.OPTIMAL == so.status
    assert sg.rel_kkt <= 1e-4
    assert abs(sg.primal_obj - so.primal_obj) <= TOL_OBJ * (1 + abs(so.primal_obj))
    assert abs(sg.dual_obj - so.dual_obj) <= TOL_OBJ * (1 + abs(so.dual_obj))
    assert sg.iterations == so.iterations and sg.restarts == so.restarts and sg.returned_average == so.returned_average
    k = oracle.kkt_unscaled(lp, sg.x, sg.y)              # the returned point really has that KKT error
    assert k["rel_kkt"] == pytest.approx(sg.rel_kkt, rel=1e-6, abs=1e-12)
    assert k["pobj"] == pytest.approx(sg.primal_obj, rel=1e-9)


@pytest.mark.parametrize("i", [1, 2, 3])
def test_convergence_parity_against_stored_oracle_runs(i):
    """Configs 1-3 take the oracle 0.5 - 15 minutes: its results are stored by tests/golden/make_oracle_golden.py."""
    gold = json.load(open(os.path.join(GOLDEN, "oracle_converged.json")))[f"uc_config{i}"]
    lp = uc_config(i)
    assert (lp.m, lp.n, lp.nnz) == (gold["m"], gold["n"], gold["nnz"])
    with P.UcLp(lp) as h:
        sg = h.solve(trace_checks=4096)
    assert sg.status == P.OPTIMAL == gold["status"] and sg.rel_kkt <= 1e-4
    assert abs(sg.primal_obj - gold["primal_obj"]) <= TOL_OBJ * abs(gold["primal_obj"])
    assert abs(sg.dual_obj - gold["dual_obj"]) <= TOL_OBJ * abs(gold["dual_obj"])
    # same terminating attempt, same restarts at the same checks with the same candidates
    assert sg.iterations == gold["iterations"] and sg.accepted == gold["accepted"] and sg.restarts == gold["restarts"]
    assert sg.returned_average == gold["returned_average"]
    trace = [[int(c["k"]), int(c["restart_kind"]), int(c["candidate"])] for c in sg.checks if c["restart_kind"]]
    assert trace == gold["restart_trace"]
    assert sg.omega == pytest.approx(gold["omega"], rel=1e-9) and sg.eta == pytest.approx(gold["eta"], rel=1e-9)
    k = oracle.kkt_unscaled(lp, sg.x, sg.y)
    assert k["rel_kkt"] <= 1.0001e-4 and k["pobj"] == pytest.approx(sg.primal_obj, rel=1e-9)


def test_converged_objective_matches_highs_on_config1():
    lp = uc_config(1)
    obj, _, _ = highs(lp)
    with P.UcLp(lp) as h:
        sg = h.solve()
    assert abs(sg.primal_obj - obj) <= 1e-3 * (1 + abs(obj))


# ------------------------------------------------------------------ full sizes of BASELINE.json
def test_paper_scale_config3_trajectory_parity():
    """Config 3 (6,049 buses, T=96) in the launch configuration bench.py times: 200 fixed attempts,
    every element of x and y compared (the oracle needs ~0.1 s per attempt at this size)."""
    sg, so = assert_trajectory_parity(uc_config(3), 200)
    assert so.restarts >= 1


@pytest.mark.parametrize("seed,F", [(10, 200), (11, 200), (12, 64)])
def test_roofline_sweep_parity(seed, F):
    from workloads import sweep_config
    assert_trajectory_parity(sweep_config(seed), F)


@pytest.mark.parametrize("seed", [12, 13, 14])
def test_roofline_sweep_parity_200_attempts_against_stored_oracle(seed):
    """BASELINE.json configs[4] at the 200 fixed attempts north_star states, m = n = 4e6 / 1e7 / 2e7 (checks and restarts
    at k = 64, 128, 192 run at full size).  The oracle needs 3 / 11 / 25 minutes there, so its run is stored by
    tests/golden/make_sweep_golden.py (oracle/ + workloads/ only): the full per-attempt trace -- every record holds
    three reductions over ALL entries of the iterate --, the check trace, norms, seeded sample positions and seeded
    random projections of x and y."""
    from workloads import sweep_config
    path = os.path.join(GOLDEN, f"oracle_sweep_seed{seed}.json")
    gold = json.load(open(path))
    lp = sweep_config(seed)
    assert (lp.m, lp.n, lp.nnz) == (gold["m"], gold["n"], gold["nnz"])
    F = gold["fixed_iterations"]
    assert F == 200
    with P.UcLp(lp) as h:
        sg = h.solve(fixed_iterations=F, trace_attempts=F, trace_checks=64)
    assert sg.iterations == F == gold["iterations"] and sg.accepted == gold["accepted"] and sg.restarts == gold["restarts"]
    ga = gold["attempts"]
    np.testing.assert_array_equal(sg.attempts["accepted"], np.array(ga["accepted"]))
    for key in ("eta_used", "eta_next", "dx2", "dy2", "inter"):
        np.testing.assert_allclose(sg.attempts[key], np.array(ga[key]), rtol=1e-9, atol=0, err_msg=key)
    assert len(sg.checks) == len(gold["checks"]) == 3
    for c, g in zip(sg.checks, gold["checks"]):
        assert (int(c["k"]), int(c["restart_kind"]), int(c["candidate"])) == (g["k"], g["restart_kind"], g["candidate"])
        assert c["omega_after"] == pytest.approx(g["omega_after"], rel=1e-9)
        assert c["mu_c"] == pytest.approx(g["mu_c"], rel=1e-8) and c["mu_r"] == pytest.approx(g["mu_r"], rel=1e-8)
    # sampled outputs: relative L2 over the sample, against the norm of the oracle's sample
    ix, iy = np.array(gold["x_pos"]), np.array(gold["y_pos"])
    assert rel_l2(sg.x[ix], np.array(gold["x_val"])) <= TOL_ITER
    assert rel_l2(sg.y[iy], np.array(gold["y_val"])) <= TOL_ITER
    assert np.linalg.norm(sg.x) == pytest.approx(gold["x_norm"], rel=1e-10)
    assert np.linalg.norm(sg.y) == pytest.approx(gold["y_norm"], rel=1e-10)
    # random projections r.x, s.y with r, s ~ N(0,1): |r.(x - x_o)| <= ~|x - x_o|, so 1e-10 |x| bounds the difference
    for q in range(len(gold["x_proj"])):
        for v, which, ref, nrm in ((sg.x, 0, gold["x_proj"][q], gold["x_norm"]), (sg.y, 1, gold["y_proj"][q], gold["y_norm"])):
            rng = np.random.default_rng(777 + 10 * q + which)
            acc = 0.0
            for s_ in range(0, v.size, 1 << 22):
                r = rng.standard_normal(min(1 << 22, v.size - s_))
                acc += float(np.sum((r * v[s_:s_ + r.size]).astype(np.longdouble)))
            assert abs(acc - ref) <= 5e-10 * nrm, (q, which)
    assert sg.eta == pytest.approx(gold["eta"], rel=1e-9) and sg.omega == pytest.approx(gold["omega"], rel=1e-9)
    assert sg.primal_obj == pytest.approx(gold["primal_obj"], rel=1e-9)


def _host_gb():
    try:
        import psutil
        return psutil.virtual_memory().available / 2**30
    except Exception:
        return 0.0


@pytest.mark.skipif(_host_gb() < 48 and not os.environ.get("UC_PDHG_BIG"),
                    reason="m = n = 1e7 / 2e7 (BASELINE.json configs[4], the two largest sizes): needs ~25 GB of host RAM "
                           "for the generator + oracle; set UC_PDHG_BIG=1 to force")
@pytest.mark.parametrize("seed,F", [(13, 16), (14, 8)])
def test_roofline_sweep_parity_largest(seed, F):
    """~1 and ~1.5 minutes (generator + oracle on one host core); full-size parity of the roofline sweep."""
    from workloads import sweep_config
    assert_trajectory_parity(sweep_config(seed), F)


# ------------------------------------------------------------------ degenerate inputs
def test_empty_problem_and_no_columns():
    z = np.zeros(0)
    lp = LP(m=0, n=0, row_ptr=np.zeros(1, np.int64), col_idx=np.zeros(0, np.int32), val=z, sense=np.zeros(0, np.uint8),
            b=z, c=z, l=z, u=z)
    with P.UcLp(lp) as h:
        s = h.solve(fixed_iterations=5)
        assert s.iterations == 5 and s.x.size == 0
        s = h.solve()
        assert s.status == P.OPTIMAL
    lp = LP(m=2, n=0, row_ptr=np.zeros(3, np.int64), col_idx=np.zeros(0, np.int32), val=z,
            sense=np.full(2, ord("G"), np.uint8), b=-np.ones(2), c=z, l=z, u=z)
    so = oracle.solve(lp, fixed_iterations=70)
    with P.UcLp(lp) as h:
        s = h.solve(fixed_iterations=70)
    np.testing.assert_array_equal(s.y, so.y)


def test_box_only_closed_form():
    lp = tiny.box_only(n=40, seed=3)
    with P.UcLp(lp) as h:
        s = h.solve(eps_rel=1e-9, eps_abs=1e-9)         # at the default 1e-4 the point is only 1e-4-close to the vertex
    expect = np.where(lp.c > 0, lp.l, np.where(lp.c < 0, lp.u, np.clip(0.0, lp.l, lp.u)))
    assert s.status == P.OPTIMAL
    np.testing.assert_allclose(s.x, expect, atol=1e-9)


def test_iteration_limit_returns_best_of_current_and_average():
    lp = get_lp("uc0")
    so = oracle.solve(lp, iter_limit=100)
    with P.UcLp(lp) as h:
        sg = h.solve(iter_limit=100)
    assert sg.status == P.ITERATION_LIMIT == so.status and sg.iterations == 100
    assert sg.returned_average == so.returned_average
    assert rel_l2(sg.x, so.x) <= TOL_ITER and rel_l2(sg.y, so.y) <= TOL_ITER
    assert sg.rel_kkt == pytest.approx(so.rel_kkt, rel=1e-6)


def test_fixed_commitment_resolve_with_update_bounds():
    lp = get_lp("uc0")
    G, T, V, oU = lp.meta["G"], lp.meta["T"], lp.meta["V"], lp.meta["offsets"]["u"]
    with P.UcLp(lp) as h:
        relaxed = h.solve()
        pattern = (relaxed.x.reshape(T, V)[:, oU:oU + G].T > 0.5).astype(float)
        fixed = fix_commitment(lp, pattern)
        so = oracle.solve(fixed)
        h.update_bounds(fixed.l, fixed.u)
        sg = h.solve()
        h.update_bounds(lp.l, lp.u)
        again = h.solve()
    assert sg.status == P.OPTIMAL
    assert abs(sg.primal_obj - so.primal_obj) <= TOL_OBJ * (1 + abs(so.primal_obj))
    assert sg.iterations == so.iterations
    assert sg.primal_obj >= relaxed.primal_obj * (1 - 2e-4)          # fixing u cannot improve the optimum
    assert again.iterations == relaxed.iterations and again.primal_obj == relaxed.primal_obj


def test_warm_started_fixed_commitment_resolve_matches_oracle():
    """SURVEY.md 8(f) NEXT-2 (P:l.60 "relaxed", l.62 re-solves): fix the commitment with uc_lp_update_bounds and re-solve
    FROM THE PREVIOUS (x, y); the oracle does the same on the fixed LP with the same warm start."""
    lp = get_lp("uc0")
    G, T, V, oU = lp.meta["G"], lp.meta["T"], lp.meta["V"], lp.meta["offsets"]["u"]
    with P.UcLp(lp) as h:
        relaxed = h.solve()
        pattern = (relaxed.x.reshape(T, V)[:, oU:oU + G].T > 0.5).astype(float)
        fixed = fix_commitment(lp, pattern)
        h.update_bounds(fixed.l, fixed.u)
        cold = h.solve(trace_checks=4096)
        warm = h.solve(x0=relaxed.x, y0=relaxed.y, trace_checks=4096)
        warm200 = h.solve(x0=relaxed.x, y0=relaxed.y, fixed_iterations=200)
    so = oracle.solve(fixed, x0=relaxed.x, y0=relaxed.y)
    so200 = oracle.solve(fixed, x0=relaxed.x, y0=relaxed.y, fixed_iterations=200)
    assert warm.status == P.OPTIMAL == so.status and warm.iterations == so.iterations and warm.restarts == so.restarts
    assert abs(warm.primal_obj - so.primal_obj) <= TOL_OBJ * (1 + abs(so.primal_obj))
    np.testing.assert_array_equal(warm.checks["restart_kind"], so.checks["restart_kind"])
    assert rel_l2(warm200.x, so200.x) <= TOL_ITER and rel_l2(warm200.y, so200.y) <= TOL_ITER
    assert abs(warm.primal_obj - cold.primal_obj) <= 2e-4 * (1 + abs(cold.primal_obj))      # same LP, both at 1e-4
    assert warm.iterations <= cold.iterations


@pytest.mark.parametrize("name", ["uc0", "uc1"])
def test_resolve_that_carries_step_size_and_primal_weight_matches_oracle(name):
    """DESIGN.md R2b: a branch-and-bound style child -- commitments the relaxation left integral are
    fixed with uc_lp_update_bounds -- re-solved from the parent's (x, y) AND its final eta, omega.  The oracle is given the
    same child LP, point and state: same trajectory for 200 attempts, same attempt count and restart trace at 1e-4."""
    import copy
    lp = get_lp(name)
    G, T, V, oU = lp.meta["G"], lp.meta["T"], lp.meta["V"], lp.meta["offsets"]["u"]
    with P.UcLp(lp) as h:
        parent = h.solve()
        assert parent.status == P.OPTIMAL and parent.eta > 0 and parent.omega > 0
        U = parent.x.reshape(T, V)[:, oU:oU + G]
        l2 = lp.l.copy().reshape(T, V); u2 = lp.u.copy().reshape(T, V)
        l2[:, oU:oU + G][U >= 1.0 - 1e-3] = 1.0; u2[:, oU:oU + G][U <= 1e-3] = 0.0
        child = copy.copy(lp); child.l = l2.ravel(); child.u = u2.ravel()
        h.update_bounds(child.l, child.u)
        kw = dict(x0=parent.x, y0=parent.y, eta0=parent.eta, omega0=parent.omega)
        g200 = h.solve(fixed_iterations=200, trace_attempts=200, trace_checks=8, **kw)
        gconv = h.solve(trace_checks=4096, **kw)
        with pytest.raises(P.UcError):
            h.solve(eta0=-1.0)
        with pytest.raises(P.UcError):
            h.solve(omega0=float("inf"))
    o200 = oracle.solve(child, fixed_iterations=200, trace_attempts=200, trace_checks=8, **kw)
    oconv = oracle.solve(child, **kw)
    assert g200.attempts["eta_used"][0] == parent.eta == o200.attempts["eta_used"][0]
    np.testing.assert_array_equal(g200.attempts["accepted"], o200.attempts["accepted"])
    np.testing.assert_allclose(g200.attempts["eta_used"], o200.attempts["eta_used"], rtol=1e-9)
    np.testing.assert_array_equal(g200.checks["restart_kind"], o200.checks["restart_kind"])
    assert rel_l2(g200.x, o200.x) <= TOL_ITER and rel_l2(g200.y, o200.y) <= TOL_ITER
    assert g200.omega == pytest.approx(o200.omega, rel=1e-9)
    assert gconv.status == P.OPTIMAL == oconv.status and gconv.iterations == oconv.iterations and gconv.restarts == oconv.restarts
    assert abs(gconv.primal_obj - oconv.primal_obj) <= TOL_OBJ * (1 + abs(oconv.primal_obj))


def test_update_objective_equals_a_fresh_handle_and_the_oracle():
    """uc_lp_update_objective: the handle behaves like one created with the new c (the scalings do not depend on c)."""
    from workloads.lp import LP
    lp = get_lp("uc0")
    rng = np.random.default_rng(17)
    c2 = lp.c * rng.uniform(0.5, 1.5, lp.n)
    lp2 = LP(m=lp.m, n=lp.n, row_ptr=lp.row_ptr, col_idx=lp.col_idx, val=lp.val, sense=lp.sense, b=lp.b, c=c2, l=lp.l, u=lp.u)
    so = oracle.solve(lp2, fixed_iterations=200, trace_attempts=200)
    with P.UcLp(lp) as h:
        first = h.solve(fixed_iterations=200)
        h.update_objective(c2)
        sg = h.solve(fixed_iterations=200, trace_attempts=200)
        conv = h.solve()
        h.update_objective(lp.c)
        back = h.solve(fixed_iterations=200)
        with pytest.raises(P.UcError):
            h.update_objective(np.full(lp.n, np.nan))
    with P.UcLp(lp2) as h2:
        fresh = h2.solve(fixed_iterations=200)
    np.testing.assert_array_equal(sg.x, fresh.x); np.testing.assert_array_equal(sg.y, fresh.y)
    np.testing.assert_array_equal(back.x, first.x); np.testing.assert_array_equal(back.y, first.y)
    np.testing.assert_array_equal(sg.attempts["accepted"], so.attempts["accepted"])
    assert rel_l2(sg.x, so.x) <= TOL_ITER and rel_l2(sg.y, so.y) <= TOL_ITER
    oc = oracle.solve(lp2)
    assert conv.status == P.OPTIMAL and conv.iterations == oc.iterations
    assert abs(conv.primal_obj - oc.primal_obj) <= TOL_OBJ * (1 + abs(oc.primal_obj))


def test_solves_are_reproducible_bit_for_bit():
    lp = get_lp("uc1")
    with P.UcLp(lp) as h:
        a = h.solve(fixed_iterations=300)
        b = h.solve(fixed_iterations=300)
    with P.UcLp(lp) as h2:
        c = h2.solve(fixed_iterations=300)
    np.testing.assert_array_equal(a.x, b.x); np.testing.assert_array_equal(a.y, b.y)
    np.testing.assert_array_equal(a.x, c.x); np.testing.assert_array_equal(a.y, c.y)


def test_long_run_crosses_step_rule_table_growth():
    """The {(k+1)^-0.6, (k+1)^-0.3} table of R5 starts at 2^18 entries and is doubled by the launch loop while the
    solve is in flight: 300,000 attempts cross that switch; the step sizes must stay those of the oracle."""
    lp = uc_config(0)
    F = 300_000
    so = oracle.solve(lp, fixed_iterations=F, trace_attempts=F)
    with P.UcLp(lp) as h:
        sg = h.solve(fixed_iterations=F, trace_attempts=F)
    assert sg.iterations == so.iterations == F
    assert np.array_equal(sg.attempts["accepted"], so.attempts["accepted"])
    assert np.array_equal(sg.attempts["eta_next"][-1000:], so.attempts["eta_next"][-1000:])
    assert rel_l2(sg.x, so.x) <= 1e-10 and rel_l2(sg.y, so.y) <= 1e-10
