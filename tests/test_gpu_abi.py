"""ABI behaviour on a GPU (-m gpu): cancel ("Terminate the other solver"), busy handle,
time limit, device-pointer entry point, the paper's stopping knobs."""
import threading
import time

import numpy as np
import pytest

import oracle
import paper_2607_03627_b200 as P
from workloads import uc_config

from helpers import rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lp1():
    return uc_config(1)


def test_cancel_before_solve_is_not_lost(lp1):
    with P.UcLp(lp1) as h:
        h.cancel()
        s = h.solve()
        assert s.status == P.CANCELLED and s.iterations == 0
        s = h.solve(fixed_iterations=64)                  # flag was consumed: the handle is reusable
        assert s.status == P.ITERATION_LIMIT and s.iterations == 64


def test_cancel_from_another_thread_stops_within_a_few_checks(lp1):
    with P.UcLp(lp1) as h:
        ref = h.solve(fixed_iterations=64 * 40)            # measure the pace: seconds per check block
        per_block = ref.loop_seconds / 40
        out = {}

        def run():
            out["s"] = h.solve(iter_limit=10_000_000, eps_rel=0.0, eps_abs=0.0)

        t = threading.Thread(target=run)
        t.start()
        time.sleep(0.2)
        with pytest.raises(P.UcError) as e:                # a second solve on the same handle is refused
            h.solve(fixed_iterations=1)
        assert e.value.code == -4
        t0 = time.time()
        h.cancel()
        t.join(timeout=30)
        latency = time.time() - t0
        assert not t.is_alive()
        s = out["s"]
        assert s.status == P.CANCELLED and s.iterations % 64 == 0 and s.iterations > 0
        assert latency < max(0.25, 20 * per_block)         # far below the 0.5 s poll of Algorithm 1
        again = h.solve(fixed_iterations=64)               # handle reusable, flag cleared
        assert again.status == P.ITERATION_LIMIT


def test_cancel_clear_drops_a_request_sent_after_the_solve_returned(lp1):
    with P.UcLp(lp1) as h:
        assert h.solve(fixed_iterations=64).status == P.ITERATION_LIMIT
        assert h.cancel_clear() is False                   # nothing pending
        h.cancel()                                         # too late for that solve: kept for the next one ...
        assert h.cancel_clear() is True                    # ... unless the caller says it was meant for the last one
        s = h.solve(fixed_iterations=64)
        assert s.status == P.ITERATION_LIMIT and s.iterations == 64


def test_release_scratch_frees_the_cached_create_block_and_create_still_works(lp1):
    with P.UcLp(lp1) as h:
        held = h.info().scratch_cached_bytes
        assert held > 0                                    # uc_lp_create keeps its scratch block for the next create
        ref = h.solve(fixed_iterations=64)
        assert P.release_scratch(-1) == held
        assert h.info().scratch_cached_bytes == 0 and P.release_scratch(-1) == 0
        with P.UcLp(lp1) as h2:                            # allocates again, same result
            again = h2.solve(fixed_iterations=64)
            assert h2.info().scratch_cached_bytes > 0
        assert np.array_equal(ref.x, again.x) and np.array_equal(ref.y, again.y)


def test_create_rejected_after_its_copies_were_enqueued_leaves_the_scratch_cache_usable(lp1):
    """A duplicate entry is found by the validation thread while the H2D copies of the CSR are already enqueued on the
    handle's stream; the scratch block must not go back to the cache (and to the next create) before they are done."""
    bad_cols = lp1.col_idx.copy()
    r0 = int(np.argmax(np.diff(lp1.row_ptr) >= 2)); p0 = int(lp1.row_ptr[r0])
    bad_cols[p0 + 1] = bad_cols[p0]                        # duplicate (row, col)
    import copy
    bad = copy.copy(lp1); bad.col_idx = bad_cols
    for _ in range(3):
        with pytest.raises(P.UcError) as e:
            P.UcLp(bad)
        assert e.value.code == -1
        with P.UcLp(lp1) as h:
            h.uc_lp_compare_layout(lp1)                       # what the device holds is the good LP's layout, bit for bit
            assert h.solve(fixed_iterations=64).iterations == 64


def test_time_limit(lp1):
    with P.UcLp(lp1) as h:
        s = h.solve(iter_limit=50_000_000, eps_rel=0.0, eps_abs=0.0, time_limit_s=0.3)
        assert s.status == P.TIME_LIMIT and 0.25 < s.solve_seconds < 3.0


def test_paper_stopping_knobs(lp1):
    """iteration limit 100,000, absolute feasibility tolerance 1e-5, convergence tolerance 1e-4."""
    p = P.default_params()
    assert p.iter_limit == 100000 and p.eps_rel == 1e-4 and p.check_every == 64
    lp = uc_config(0)
    with P.UcLp(lp) as h:
        loose = h.solve()
        tight = h.solve(eps_abs=1e-5)
    so = oracle.solve(lp, eps_abs=1e-5)
    assert tight.status == P.OPTIMAL and tight.iterations >= loose.iterations
    assert tight.iterations == so.iterations


def test_device_pointer_entry_point_with_torch_memory_and_stream(lp1):
    import torch
    dev = torch.device("cuda:0")
    x = torch.empty(lp1.n, dtype=torch.float64, device=dev)
    y = torch.empty(lp1.m, dtype=torch.float64, device=dev)
    stream = torch.cuda.Stream()
    with P.UcLp(lp1) as h:
        host = h.solve(fixed_iterations=128)
        with torch.cuda.stream(stream):
            s = h.solve_device(x, y, fixed_iterations=128, stream=stream.cuda_stream)
        stream.synchronize()
        np.testing.assert_array_equal(x.cpu().numpy(), host.x)
        np.testing.assert_array_equal(y.cpu().numpy(), host.y)
        # warm start from device tensors: continue 72 more attempts is NOT the same trajectory (state resets), but it must run
        s2 = h.solve_device(x, y, x0=x.clone(), y0=y.clone(), fixed_iterations=8, stream=stream.cuda_stream)
        assert s2.iterations == 8 and s.kernel_launches > 2 * 128


def test_info_and_launch_count(lp1):
    with P.UcLp(lp1) as h:
        i = h.info()
        assert (i.m, i.n, i.nnz) == (lp1.m, lp1.n, lp1.nnz)
        assert i.k_sell_slots + i.k_long_nnz >= lp1.nnz and i.kt_sell_slots + i.kt_long_nnz >= lp1.nnz
        assert i.k_long_rows == lp1.meta["T"]                      # the T reserve rows (G = 90 entries) form the long tail
        assert (i.k_sell_slots + i.k_long_nnz) / lp1.nnz < 1.03    # sliced-ELL padding stays below 3 %
        assert i.bytes_per_attempt > 24 * lp1.nnz
        s = h.solve(fixed_iterations=128)
        assert s.kernel_launches >= 2 * 128 + 2 * 5


def test_different_handles_solve_concurrently_on_their_own_streams(lp1):
    """include/uc_pdhg.h: the call is not re-entrant per handle, but different handles may solve at the same time
    (the paper's 45 scenarios are independent LPs).  Results must be those of a solve run alone."""
    with P.UcLp(lp1) as h0:
        alone = h0.solve(fixed_iterations=640)
    handles = [P.UcLp(lp1) for _ in range(3)]
    out = [None] * 3

    def run(i):
        out[i] = handles[i].solve(fixed_iterations=640)

    try:
        th = [threading.Thread(target=run, args=(i,)) for i in range(3)]
        [t.start() for t in th]
        [t.join(timeout=120) for t in th]
        assert not any(t.is_alive() for t in th)
        for s in out:
            assert s.status == P.ITERATION_LIMIT and s.iterations == 640
            assert np.array_equal(s.x, alone.x) and np.array_equal(s.y, alone.y)
    finally:
        for h in handles:
            h.close()


def test_solve_batch_results_are_those_of_solo_solves(lp1):
    """uc_pdhg_solve_batch (the paper's 45 scenarios, P:l.101): different LPs solved concurrently
    inside one call, fewer workers than handles; every result is bit-identical to the solve run alone."""
    lps = [uc_config(0), lp1, uc_config("tuned_presolve"), uc_config(0), lp1, uc_config("tuned_presolve"), uc_config(0)]
    handles = [P.UcLp(lp) for lp in lps]
    try:
        solo = [h.solve(fixed_iterations=320) for h in handles[:3]]
        out = P.solve_batch(handles, max_concurrent=3, fixed_iterations=320)
        assert len(out) == len(handles)
        for i, s in enumerate(out):
            assert s.status == P.ITERATION_LIMIT and s.iterations == 320
            assert np.array_equal(s.x, solo[i % 3].x) and np.array_equal(s.y, solo[i % 3].y)
        conv = P.solve_batch(handles[:3])                         # default stopping rule
        for s, h in zip(conv, handles[:3]):
            alone = h.solve()
            assert s.status == P.OPTIMAL and s.iterations == alone.iterations and s.primal_obj == alone.primal_obj
        with pytest.raises(P.UcError):
            P.solve_batch([handles[0], handles[0]])               # the same handle twice
    finally:
        for h in handles:
            h.close()


def test_results_do_not_depend_on_the_cta_limit(lp1):
    """uc_lp_options.max_ctas only changes how the slices are dealt to CTAs and warps: bit-identical iterates."""
    with P.UcLp(lp1) as a, P.UcLp(lp1, max_ctas=5) as b, P.UcLp(lp1, max_ctas=37) as c:
        sa, sb, sc = (h.solve(fixed_iterations=256, trace_attempts=256) for h in (a, b, c))
    for s in (sb, sc):
        np.testing.assert_array_equal(s.x, sa.x); np.testing.assert_array_equal(s.y, sa.y)
        np.testing.assert_array_equal(s.attempts["eta_used"], sa.attempts["eta_used"])


def test_timeline_hook_is_refused_by_the_product_build(lp1):
    with P.UcLp(lp1) as h:
        with pytest.raises(P.UcError) as e:
            h.timeline(4)
    assert "UC_TIMELINE" in str(e.value)
