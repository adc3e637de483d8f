"""Algorithm 1 of the paper: race the GPU PDHG solver against a CPU LP solver on the same
relaxed problem and terminate the loser.

    1  partition the CPU cores between the two pipelines                     (l.70; here: `cpu_cores`, `gpu_host_cores`)
    2  start pipeline 1: PDHG on the GPU                                      (l.74)
    3  start pipeline 2: the CPU competitor                                   (l.77)
    4  while neither has converged: sleep `poll_s` (0.5 s in the paper, l.81)
    5  terminate the other solver, return the winner's solution               (l.82-85)

The paper's competitor is Gurobi's barrier; it is not available here, so the competitor is any callable that
solves the LP on the host (the tests use HiGHS through scipy).  It runs in a child PROCESS, because "terminate"
has to work on a solver that offers no cancel hook; the GPU side is stopped with uc_pdhg_cancel, which is what
that entry point exists for.  Crossover, simplex clean-up and branch-and-bound (the rest of both pipelines) are
out of scope.
"""
from __future__ import annotations

import multiprocessing as mp
import os
import threading
import time
from dataclasses import dataclass, field
from typing import Any, Callable, Optional

from . import binding as _b


@dataclass
class RaceResult:
    winner: str                      # "gpu_pdhg" or "cpu"
    objective: float
    seconds: float                   # wall time until the winner was seen (poll granularity included)
    gpu: Optional[Any] = None        # Solution of the GPU side (status CANCELLED if it lost)
    cpu: Optional[Any] = None        # whatever the competitor returned (None if it was terminated)
    gpu_seconds: Optional[float] = None      # when the GPU side returned, from the start of the race
    cpu_seconds: Optional[float] = None      # when the competitor returned (None if terminated)
    cancel_latency_s: Optional[float] = None  # uc_pdhg_cancel -> uc_pdhg_solve returned (only if the GPU lost)
    polls: int = 0
    log: list = field(default_factory=list)


def partition_cores(total: Optional[int] = None):
    """Line 1 of Algorithm 1 ("Partition 48 CPU cores evenly between two solver instances"): the cores
    this process may run on, split evenly -- (cores of the GPU pipeline's host thread, cores of the CPU competitor).
    With fewer than two cores both sides get everything."""
    try:
        avail = sorted(os.sched_getaffinity(0))
    except AttributeError:                      # not Linux
        avail = list(range(os.cpu_count() or 1))
    if total is not None:
        avail = avail[:max(1, int(total))]
    if len(avail) < 2:
        return set(avail), set(avail)
    half = len(avail) // 2
    return set(avail[:half]), set(avail[half:])


def _child(fn, args, q, cores):
    try:
        if cores:
            try:
                os.sched_setaffinity(0, cores)          # the competitor's threads inherit it
                os.environ["OMP_NUM_THREADS"] = str(len(cores))
            except (AttributeError, OSError):
                pass
        q.put(("ok", fn(*args)))
    except BaseException as e:      # the parent must never wait for a dead child
        q.put(("error", repr(e)))


def race(handle: "_b.UcLp", competitor: Callable[..., Any], competitor_args: tuple = (), *,
         competitor_objective: Callable[[Any], float] = lambda r: float(r),
         poll_s: float = 0.5, solve_kwargs: Optional[dict] = None, mp_context: str = "fork",
         cpu_cores: Optional[set] = None, gpu_host_cores: Optional[set] = None) -> RaceResult:
    """Run Algorithm 1.  `handle` is a created UcLp (the LP is already on the GPU: presolve and model building
    are upstream of this library); `competitor(*competitor_args)` solves the same LP on the host and returns
    something `competitor_objective` can turn into the optimal objective value.
    `cpu_cores` / `gpu_host_cores` (line 1, P:l.70): CPU sets the competitor process and the thread that drives
    uc_pdhg_solve are pinned to (os.sched_setaffinity); None = no pinning; `partition_cores()` gives the paper's
    even split.  The loop ends when the GPU side returns OPTIMAL, when the competitor returns a solution, or when
    both have finished; a GPU return with any other status (iteration limit, time limit, numerical error) is logged
    and the competitor is waited for ("while neither has converged", P:l.80)."""
    solve_kwargs = dict(solve_kwargs or {})
    t0 = time.perf_counter()
    box: dict = {}

    def gpu_side():
        if gpu_host_cores:
            try:
                os.sched_setaffinity(threading.get_native_id(), gpu_host_cores)
            except (AttributeError, OSError):
                pass
        try:
            box["sol"] = handle.solve(**solve_kwargs)
        except BaseException as e:      # the poll loop must never wait for a dead thread
            box["error"] = repr(e)
        box["t"] = time.perf_counter() - t0

    ctx = mp.get_context(mp_context)
    q = ctx.Queue()
    proc = ctx.Process(target=_child, args=(competitor, competitor_args, q, cpu_cores), daemon=True)
    th = threading.Thread(target=gpu_side, daemon=True)
    th.start()                       # line 2: pipeline 1
    proc.start()                     # line 3: pipeline 2
    res = RaceResult(winner="", objective=float("nan"), seconds=0.0)
    cpu_msg = None
    gpu_logged = False
    while True:                      # line 4: while neither has converged
        gpu_done = not th.is_alive()
        if cpu_msg is None and not q.empty():
            cpu_msg = q.get()
            res.cpu_seconds = time.perf_counter() - t0
        gpu_conv = gpu_done and box.get("sol") is not None and box["sol"].status == _b.OPTIMAL
        cpu_conv = cpu_msg is not None and cpu_msg[0] == "ok"
        cpu_done = cpu_msg is not None or not proc.is_alive()
        if gpu_conv or cpu_conv or (gpu_done and cpu_done):
            if cpu_msg is None and not q.empty():                   # the child put its message just before exiting
                cpu_msg = q.get()
                res.cpu_seconds = time.perf_counter() - t0
            break
        if gpu_done and not gpu_logged:                             # keep waiting for the competitor
            gpu_logged = True
            st = box["sol"].status if box.get("sol") is not None else None
            res.log.append("gpu side returned without converging: " +
                           (_b.STATUS_NAMES.get(st, str(st)) if st is not None else box.get("error", "no result")))
        if cpu_msg is not None and cpu_msg[0] == "error" and "competitor failed" not in " ".join(res.log):
            res.log.append("competitor failed: " + cpu_msg[1])     # keep waiting for the GPU side
        time.sleep(poll_s)
        res.polls += 1
    res.seconds = time.perf_counter() - t0
    gpu_ok = (not th.is_alive()) and box.get("sol") is not None and box["sol"].status == _b.OPTIMAL
    cpu_ok = cpu_msg is not None and cpu_msg[0] == "ok"
    if gpu_ok and (not cpu_ok or box["t"] <= (res.cpu_seconds or float("inf"))):
        # line 5, GPU first: terminate the competitor
        res.winner = "gpu_pdhg"
        res.objective = box["sol"].primal_obj
        if proc.is_alive():
            proc.terminate()
        res.log.append("competitor terminated")
    elif cpu_ok:
        # line 5, CPU first: stop the GPU solver through its cancel hook and time how long it takes to return
        res.winner = "cpu"
        res.cpu = cpu_msg[1]
        res.objective = competitor_objective(cpu_msg[1])
        if th.is_alive():
            tc = time.perf_counter()
            handle.cancel()
            th.join()
            res.cancel_latency_s = time.perf_counter() - tc
            res.log.append("uc_pdhg_cancel sent")
            # The thread being alive does not mean the library is still inside the solve: a cancel that lands after the
            # solve has left its loop is kept for the NEXT solve on the handle (uc_pdhg.h), and callers reuse handles
            # (re-solves, the "GPU alone" column of _main).  The solve returned on its own, so drop that request.
            sol = box.get("sol")
            if (sol is None or sol.status != _b.CANCELLED) and hasattr(handle, "cancel_clear") and handle.cancel_clear():
                res.log.append("cancel arrived after the GPU solve had returned: request dropped")
    else:
        th.join()
        if proc.is_alive():
            proc.terminate()
        proc.join(timeout=5.0)
        raise RuntimeError(f"neither solver converged: gpu {box.get('sol') or box.get('error')}, cpu {cpu_msg}")
    proc.join(timeout=5.0)
    if th.is_alive():
        th.join()
    res.gpu = box.get("sol")
    res.gpu_seconds = box.get("t")
    return res


def highs_competitor(lp, time_limit=None):
    """Stand-in for the paper's CPU barrier solver: HiGHS through scipy (optional dependency).  Returns the optimal
    objective of min c'x s.t. Ax {=,>=} b, l <= x <= u; raises if HiGHS stops for any other reason (`time_limit` s)."""
    import numpy as np
    import scipy.sparse as sp
    from scipy.optimize import linprog
    A = sp.csr_matrix((lp.val, lp.col_idx, lp.row_ptr), shape=(lp.m, lp.n))
    E = np.asarray(lp.sense) == ord("E")
    G = ~E
    bounds = [(None if np.isinf(a) else a, None if np.isinf(b) else b) for a, b in zip(lp.l, lp.u)]
    kw = {}
    if G.any():
        kw.update(A_ub=-A[G], b_ub=-lp.b[G])
    if E.any():
        kw.update(A_eq=A[E], b_eq=lp.b[E])
    r = linprog(lp.c, bounds=bounds, method="highs", options=({"time_limit": float(time_limit)} if time_limit else None), **kw)
    if r.status != 0:
        raise RuntimeError(r.message)
    return float(r.fun)


def cancel_latency(handle, after_s: float = 0.2, repeats: int = 5, **solve_kwargs):
    """Seconds between uc_pdhg_cancel and the return of a uc_pdhg_solve that is in full flight (`after_s` after its
    start, with tolerances it cannot reach): what Algorithm 1's "terminate the other solver" (P:l.82-84) costs on the
    GPU side.  Returns the list of measured latencies and the attempts each cancelled solve had run."""
    lat, its = [], []
    for _ in range(repeats):
        box = {}
        th = threading.Thread(target=lambda: box.update(sol=handle.solve(eps_rel=0.0, eps_abs=0.0, iter_limit=10**9, **solve_kwargs)), daemon=True)
        th.start()
        time.sleep(after_s)
        t = time.perf_counter()
        handle.cancel()
        th.join()
        lat.append(time.perf_counter() - t)
        assert box["sol"].status == _b.CANCELLED, _b.STATUS_NAMES.get(box["sol"].status)
        its.append(box["sol"].iterations)
    return lat, its


def _main():
    """python -m paper_2607_03627_b200.race --configs 0 1 2 tuned_presolve [--poll 0.5] [--eps-abs 1e-4 1e-5] [--cancel-config 3]:
    a Table-VI-style row per UC config and tolerance (which pipeline wins, P:l.221-226), with the CPU cores split evenly
    between the two pipelines (P:l.70), then the cancel latency of a solve in full flight."""
    import argparse
    from workloads import uc_config
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=lambda v: int(v) if v.lstrip("-").isdigit() else v, nargs="+", default=[0, 1],
                    help="UC configs of BASELINE.json (0-3) or a named shape of workloads.uc_lp (tuned_presolve: the LP size the "
                         "paper's tuned presolve leaves, P:l.232, the regime of Table VI)")
    ap.add_argument("--poll", type=float, default=0.5, help="poll period in s (0.5 in the paper, P:l.81)")
    ap.add_argument("--eps-abs", type=float, nargs="+", default=[1e-4], help="absolute tolerance(s); 1e-5 is the paper's knob (P:l.66)")
    ap.add_argument("--cancel-config", type=int, default=None)
    ap.add_argument("--alone-limit-s", type=float, default=120.0, help="time limit of the stand-alone HiGHS run of the table")
    args = ap.parse_args()
    gpu_cores, cpu_cores = partition_cores()
    print(f"cores: GPU pipeline host thread {len(gpu_cores)}, CPU competitor {len(cpu_cores)}; poll {args.poll} s")
    print("| config | eps_abs | winner | race s | GPU PDHG alone s (attempts) | HiGHS alone s | objective | cancel latency ms |")
    print("|---|---|---|---|---|---|---|---|")
    for c in args.configs:
        lp = uc_config(c)
        t = time.perf_counter()
        try:
            highs_competitor(lp, args.alone_limit_s); tcs = f"{time.perf_counter() - t:.2f}"
        except RuntimeError:
            tcs = f"> {args.alone_limit_s:g} (time limit)"
        with _b.UcLp(lp) as h:
            h.solve(fixed_iterations=64)                  # warm-up: graph instantiation is not part of the race
            for ea in args.eps_abs:
                kw = dict(eps_abs=ea)
                r = race(h, highs_competitor, (lp,), poll_s=args.poll, solve_kwargs=kw, cpu_cores=cpu_cores, gpu_host_cores=gpu_cores)
                t = time.perf_counter(); s = h.solve(**kw); tg = time.perf_counter() - t
                lat = "-" if r.cancel_latency_s is None else f"{1e3 * r.cancel_latency_s:.1f}"
                print(f"| {c} | {ea:g} | {r.winner} | {r.seconds:.2f} | {tg:.3f} ({s.iterations}) | {tcs} | {r.objective:.4f} | {lat} |", flush=True)
    if args.cancel_config is not None:
        lp = uc_config(args.cancel_config)
        with _b.UcLp(lp) as h:
            h.solve(fixed_iterations=64)
            lat, its = cancel_latency(h)
        print()
        print(f"cancel latency on config {args.cancel_config} (solve in full flight, cancelled 0.2 s after its start): "
              + ", ".join(f"{1e3 * v:.1f}" for v in lat) + f" ms; attempts run: {its}")


if __name__ == "__main__":
    _main()
