"""Algorithm 1 of the paper: the racing driver of paper_2607_03627_b200/race.py.
CPU tests drive its control flow with a stand-in for the GPU handle; the GPU test races the real PDHG solver
against HiGHS (the stand-in for the paper's barrier solver, which is not available) on UC config 1."""
import threading
import time
from types import SimpleNamespace

import numpy as np
import pytest

import paper_2607_03627_b200.binding as B
from paper_2607_03627_b200.race import race


class StandInHandle:
    """Behaves like UcLp for race(): solve() blocks for `seconds` unless cancel() arrives first."""

    def __init__(self, seconds, objective=1.25, final_status=B.OPTIMAL):
        self.seconds, self.objective, self._stop, self.cancelled = seconds, objective, threading.Event(), False
        self.final_status = final_status

    def solve(self, **kw):
        stopped = self._stop.wait(self.seconds)
        status = B.CANCELLED if stopped else self.final_status
        return SimpleNamespace(status=status, primal_obj=self.objective, iterations=0)

    def cancel(self):
        self.cancelled = True
        self._stop.set()


class LateCancelHandle(StandInHandle):
    """The window of the real library: solve() has left its loop (status decided, not CANCELLED) while its thread is still
    alive, so a cancel() sent now is parked for the next solve -- unless cancel_clear() drops it."""

    def __init__(self):
        super().__init__(seconds=0.0, final_status=B.ITERATION_LIMIT)
        self.left_loop, self.parked, self.cleared = threading.Event(), False, False

    def solve(self, **kw):
        if self.parked:                                        # what uc_pdhg_solve does with a parked request
            self.parked = False
            return SimpleNamespace(status=B.CANCELLED, primal_obj=0.0, iterations=0)
        self.left_loop.set()
        self._stop.wait(30.0)                                  # thread alive until the cancel arrives
        return SimpleNamespace(status=B.ITERATION_LIMIT, primal_obj=self.objective, iterations=64)

    def cancel(self):
        self.cancelled = self.parked = True
        self._stop.set()

    def cancel_clear(self):
        had, self.parked, self.cleared = self.parked, False, True
        return had


def slow_competitor(seconds, value):
    time.sleep(seconds)
    return value


def delayed_highs(seconds, lp):
    from helpers import highs
    time.sleep(seconds)
    return highs(lp)


def test_cpu_wins_and_the_gpu_side_is_cancelled_through_its_hook():
    h = StandInHandle(seconds=30.0)
    r = race(h, slow_competitor, (0.2, 7.5), poll_s=0.05)
    assert r.winner == "cpu" and r.objective == 7.5
    assert h.cancelled and r.gpu.status == B.CANCELLED
    assert r.cancel_latency_s is not None and r.cancel_latency_s < 1.0
    assert r.seconds < 5.0 and r.cpu_seconds is not None


def test_a_cancel_that_misses_the_solve_does_not_leak_into_the_next_one():
    h = LateCancelHandle()
    r = race(h, slow_competitor, (0.2, 7.5), poll_s=0.05)
    assert r.winner == "cpu" and h.cancelled and r.gpu.status == B.ITERATION_LIMIT
    assert h.cleared and not h.parked and any("request dropped" in m for m in r.log)
    assert h.solve().status == B.ITERATION_LIMIT               # the handle is reusable: no CANCELLED at entry


def test_gpu_wins_and_the_competitor_process_is_terminated():
    h = StandInHandle(seconds=0.2, objective=3.0)
    t0 = time.perf_counter()
    r = race(h, slow_competitor, (60.0, 9.0), poll_s=0.05)
    assert r.winner == "gpu_pdhg" and r.objective == 3.0
    assert not h.cancelled and r.cpu is None and r.cancel_latency_s is None
    assert time.perf_counter() - t0 < 10.0                 # did not wait for the 60 s competitor
    assert "competitor terminated" in r.log


def test_competitor_failure_does_not_hang_the_race():
    def broken():
        raise ValueError("no licence")
    h = StandInHandle(seconds=0.3, objective=2.0)
    r = race(h, broken, (), poll_s=0.05)
    assert r.winner == "gpu_pdhg" and r.objective == 2.0


@pytest.mark.parametrize("status", [B.ITERATION_LIMIT, B.TIME_LIMIT, B.NUMERICAL_ERROR])
def test_gpu_side_returning_early_without_converging_does_not_end_the_race(status):
    """Algorithm 1, P:l.80 "while neither has converged": a GPU return at its iteration limit is not a convergence;
    the competitor is waited for and wins."""
    h = StandInHandle(seconds=0.1, final_status=status)
    r = race(h, slow_competitor, (0.6, 4.5), poll_s=0.05)
    assert r.winner == "cpu" and r.objective == 4.5 and r.gpu.status == status
    assert not h.cancelled and r.cancel_latency_s is None            # nothing left to cancel
    assert any("without converging" in m for m in r.log)


def test_neither_converges_raises_and_leaves_no_child_behind():
    import multiprocessing as mp

    def broken():
        raise ValueError("no licence")
    h = StandInHandle(seconds=0.1, final_status=B.ITERATION_LIMIT)
    before = len(mp.active_children())
    with pytest.raises(RuntimeError, match="neither solver converged"):
        race(h, broken, (), poll_s=0.05)
    assert len(mp.active_children()) <= before


def _report_affinity():
    import os
    return sorted(os.sched_getaffinity(0))


def test_core_partition_pins_the_competitor_process():
    """Algorithm 1 line 1 (P:l.70): the cores are split evenly; the competitor process runs on its half only."""
    import os
    from paper_2607_03627_b200.race import partition_cores
    gpu_cores, cpu_cores = partition_cores()
    avail = os.sched_getaffinity(0)
    assert gpu_cores | cpu_cores == set(avail)
    if len(avail) >= 2:
        assert not (gpu_cores & cpu_cores) and abs(len(gpu_cores) - len(cpu_cores)) <= 1
    h = StandInHandle(seconds=30.0)
    r = race(h, _report_affinity, (), competitor_objective=lambda cores: float(len(cores)), poll_s=0.05,
             cpu_cores=cpu_cores, gpu_host_cores=gpu_cores)
    assert r.winner == "cpu" and r.cpu == sorted(cpu_cores)
    assert os.sched_getaffinity(0) == avail                          # the caller's own affinity is untouched


@pytest.mark.gpu
def test_race_pdhg_against_highs_both_outcomes():
    """UC config 0 (HiGHS needs ~0.3 s there; on config 1 it needs minutes, see profiles/r01d_race.md)."""
    import paper_2607_03627_b200 as P
    from helpers import highs
    from workloads import uc_config
    lp = uc_config(0)
    ref_obj, _, _ = highs(lp)
    with P.UcLp(lp) as h:
        h.solve(fixed_iterations=64)                       # warm-up: graph instantiation is not part of the race
        # default tolerances, both sides at full speed: a genuine race (PDHG ~70 ms, HiGHS ~50-350 ms here)
        r = race(h, highs, (lp,), competitor_objective=lambda out: out[0], poll_s=0.02)
        assert r.winner in ("gpu_pdhg", "cpu")
        assert abs(r.objective - ref_obj) <= 1e-3 * (1.0 + abs(ref_obj))
        # a competitor held back by 5 s: PDHG converges first and the competitor process is terminated
        t0 = time.perf_counter()
        r = race(h, delayed_highs, (5.0, lp), competitor_objective=lambda out: out[0], poll_s=0.02)
        assert r.winner == "gpu_pdhg" and r.gpu.status == P.OPTIMAL and r.gpu.rel_kkt <= 1e-4 and r.cpu is None
        assert abs(r.objective - ref_obj) <= 1e-3 * (1.0 + abs(ref_obj)) and time.perf_counter() - t0 < 4.0
        # an unreachable tolerance: HiGHS wins, the GPU solver is stopped by uc_pdhg_cancel well inside the
        # paper's 0.5 s poll period
        r = race(h, highs, (lp,), competitor_objective=lambda out: out[0], poll_s=0.02,
                 solve_kwargs=dict(eps_rel=0.0, eps_abs=0.0, iter_limit=100_000_000))
        assert r.winner == "cpu" and r.gpu.status == P.CANCELLED and r.gpu.iterations > 0
        assert abs(r.objective - ref_obj) <= 1e-9 * (1.0 + abs(ref_obj))
        assert r.cancel_latency_s < 0.5
        again = h.solve(fixed_iterations=64)               # the handle survives a race either way
        assert again.status == P.ITERATION_LIMIT and again.iterations == 64
