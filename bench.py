#!/usr/bin/env python
"""bench.py -- PDHG attempts/s on the paper-scale synthetic UC LP (BASELINE.json configs[3]) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole iteration path over the resident LP:
one uc_pdhg_solve_device call of --attempts fixed attempts (graph launches of 64 attempts + a check,
restarts included) from the initial point, inputs already in HBM.  `value` = attempts/s over all ranks
(replicas only: the path does not shard).  `e2e` = the same metric through the host-buffer
C-ABI calls: uc_lp_create from host CSR (H2D + layouts + preconditioning) -> uc_pdhg_solve to relative
KKT 1e-4 -> x, y back in host memory, i.e. attempts to converge / wall time of the whole job.
`roofline` is for the dominant kernel of an attempt, algorithmic bytes over its CUDA-event
duration; `cpu_baseline` is the oracle timed on this box's host cores on a bounded sample.
--impl reference times the CPU oracle (there is no other reference implementation: PAPER.md's solver is
closed source) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pdhg_attempts_per_s"
UNIT = "attempts/s"


def algorithmic_bytes(m, n, nnz, info=None):
    """bytes one attempt must move (fp64 values, int32 indices, both matrix copies, every
    vector once, gathers counted once).  Split by kernel; the sum is 24 nnz + 76 n + 53 m + 8.
    With `info` (uc_lp_get_info) the index bytes are those of THIS layout: 2 instead of 4 per entry in the slices that
    store 16-bit column offsets ("never credit bytes that were not moved")."""
    idx_kt = idx_k = 4.0
    if info is not None:
        idx_kt = 4.0 - 2.0 * info.kt_narrow_slots / max(info.kt_sell_slots + info.kt_long_nnz, 1)
        idx_k = 4.0 - 2.0 * info.k_narrow_slots / max(info.k_sell_slots + info.k_long_nnz, 1)
    primal = (8 + idx_kt) * nnz + 4 * (n + 1) + 64 * n + 8 * m     # K' pass: matrix, ptr, x c l u (32) + x' xbar (16) + xsum r/w (16), gather of y
    dual = (8 + idx_k) * nnz + 4 * (m + 1) + 41 * m + 8 * n        # K pass: matrix, ptr, y q sense (17) + y' (8) + ysum r/w (16), gather of xbar
    return int(primal), int(dual)


def ncu_traffic(config):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the attempt kernels, from the tracked artefact that the
    ncu summary of the same capture is written with (profiles/r02_traffic.json; bytes; cold L2 per replay)."""
    p = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        d = json.load(open(p))
        return d.get(f"uc_config{config}"), "profiles/r02_traffic.json"
    except Exception:
        return None, None


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index, period_ms=100):
        self.index, self.rows, self.proc, self.period_ms = index, [], None, int(period_ms)

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", str(self.period_ms)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_baseline(lp, budget_attempts=(10, 60)):
    """The oracle as it stands, one thread, on a bounded sample: two fixed-iteration runs, the difference
    removes its own preconditioning so that the figure is attempts/s of its loop."""
    import oracle
    a, b = budget_attempts
    t0 = time.perf_counter(); oracle.solve(lp, fixed_iterations=a); t1 = time.perf_counter()
    oracle.solve(lp, fixed_iterations=b); t2 = time.perf_counter()
    dt = (t2 - t1) - (t1 - t0)
    return {"value": (b - a) / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"config 3 ({lp.m}x{lp.n}, nnz {lp.nnz}): oracle runs of {a} and {b} fixed attempts, "
                      f"difference of wall times ({dt:.2f} s for {b - a} attempts; its setup + preconditioning {2 * (t1 - t0) - (t2 - t1) + dt:.2f} s excluded)"}


def run_reference(args, world, rank):
    """--impl reference: the CPU oracle, bounded sample per step."""
    if rank != 0:
        return
    import oracle
    from workloads import uc_config
    lp = uc_config(args.config)
    per_step = args.ref_attempts
    for _ in range(args.warmup):
        oracle.solve(lp, fixed_iterations=per_step)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.solve(lp, fixed_iterations=per_step)
    dt = time.perf_counter() - t0
    v = args.steps * per_step / dt
    sample = (f"each step = one oracle call of {per_step} fixed attempts on config {args.config} "
              f"(its own Ruiz/Pock-Chambolle preconditioning included in every call)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, lp), "attempts_per_step": per_step},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


def workload_name(i, lp):
    return f"BASELINE.json configs[{i}]: synthetic DC-UC LP {lp.name} (m={lp.m}, n={lp.n}, nnz={lp.nnz}), fp64"


def aggregate(local_seconds, local_units, dist=None, device=None):
    """Whole-job throughput: units of all ranks / max over ranks of the timed seconds (replicas only)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_seconds, local_units
    import torch
    t = torch.tensor([local_seconds], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def all_configs_table(batch_sizes=(1, 4, 16, 45)):
    """--all-configs: markdown tables over BASELINE.json's configs (UC 0-3; roofline sweep seeds 10-14 at the 200 fixed
    attempts north_star states) plus the tuned-presolve shape of PAPER.md Table VII: attempts/s of `uc_pdhg_solve_device`
    (CUDA-event loop time, checks and restarts included), and the aggregate rate of `uc_pdhg_solve_batch` on the
    launch-latency-bound LPs (the paper's 45 scenarios, P:l.101).  Reporting only: the bench line of the contract is the
    default run."""
    import numpy as np
    import torch
    import paper_2607_03627_b200 as P
    from workloads import sweep_config, uc_config
    peak, _ = load_peaks()
    st = torch.cuda.Stream()
    print("| workload | m | n | nnz | attempts | us/attempt (in graph, checks incl.) | attempts/s | algorithmic MB/attempt (this layout / 32-bit indices) | GB/s | % of measured peak | 16-bit-offset slots % | device MB | create ms |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    cases = [(f"UC config {c}", (lambda c=c: uc_config(c)), 2048) for c in (0, 1, 2, 3)]
    cases += [("UC tuned-presolve shape (P: Table VII)", (lambda: uc_config("tuned_presolve")), 2048)]
    cases += [(f"config 4, seed {s_}", (lambda s_=s_: sweep_config(s_)), 200) for s_ in (10, 11, 12, 13, 14)]
    for name, make, attempts in cases:
        lp = make()
        t = time.perf_counter(); h = P.UcLp(lp, device=0); tc = time.perf_counter() - t
        x = torch.empty(lp.n, dtype=torch.float64, device="cuda"); y = torch.empty(lp.m, dtype=torch.float64, device="cuda")
        for _ in range(2):
            r = h.solve_device(x, y, fixed_iterations=attempts, stream=st.cuda_stream)
        us = r.loop_seconds * 1e6 / attempts
        i = h.info()
        bp, bd = algorithmic_bytes(lp.m, lp.n, lp.nnz, i)
        sp, sd = algorithmic_bytes(lp.m, lp.n, lp.nnz)
        narrow = 100.0 * (i.k_narrow_slots + i.kt_narrow_slots) / max(i.k_sell_slots + i.kt_sell_slots, 1)
        print(f"| {name} | {lp.m} | {lp.n} | {lp.nnz} | {attempts} | {us:.2f} | {1e6 / us:.0f} | {(bp + bd) / 1e6:.1f} / {(sp + sd) / 1e6:.1f} | "
              f"{(bp + bd) / us / 1e3:.0f} | {(bp + bd) / us / 1e3 / peak * 100:.1f} | {narrow:.0f} | {i.device_bytes / 1e6:.0f} | {tc * 1e3:.0f} |", flush=True)
        h.close()
        del lp, x, y
    print()
    print("| workload | CTAs per kernel (max_ctas) | LPs in one uc_pdhg_solve_batch call (16 in flight) | aggregate attempts/s | per-LP attempts/s | results identical to a solo solve |")
    print("|---|---|---|---|---|---|")
    for name, key, limits in (("UC config 0", 0, (0,)), ("UC tuned-presolve shape", "tuned_presolve", (0, 37, 18)), ("UC config 1", 1, (0, 37))):
        lp = uc_config(key)
        F = 2048
        with P.UcLp(lp, device=0) as h0:
            solo = h0.solve(fixed_iterations=F)
        for lim in limits:
            hs = [P.UcLp(lp, device=0, max_ctas=lim) for _ in range(max(batch_sizes))]
            for nb in batch_sizes:
                for _ in range(2):
                    torch.cuda.synchronize(); t = time.perf_counter()
                    out = P.solve_batch(hs[:nb], fixed_iterations=F)
                    dt = time.perf_counter() - t
                same = all(np.array_equal(o.x, solo.x) and np.array_equal(o.y, solo.y) for o in out)
                print(f"| {name} | {'all SMs' if lim == 0 else lim} | {nb} | {nb * F / dt:.0f} | {F / dt:.0f} | {same} |", flush=True)
            for h in hs:
                h.close()


def sweep_line(args):
    """One size of the roofline sweep (BASELINE.json configs[4]): attempts/s and effective bandwidth of 200 fixed attempts."""
    import torch
    import paper_2607_03627_b200 as P
    from workloads import sweep_config
    lp = sweep_config(args.sweep_seed)
    peak, _ = load_peaks()
    st = torch.cuda.Stream()
    with P.UcLp(lp, device=0) as h:
        x = torch.empty(lp.n, dtype=torch.float64, device="cuda"); y = torch.empty(lp.m, dtype=torch.float64, device="cuda")
        for _ in range(max(args.warmup, 1)):
            r = h.solve_device(x, y, fixed_iterations=200, stream=st.cuda_stream)
        loop = 0.0
        for _ in range(max(args.steps, 1)):
            loop += h.solve_device(x, y, fixed_iterations=200, stream=st.cuda_stream).loop_seconds
        bp, bd = algorithmic_bytes(lp.m, lp.n, lp.nnz, h.info())
    us = loop * 1e6 / (200 * max(args.steps, 1))
    print(json.dumps({"metric": METRIC, "value": 1e6 / us, "unit": UNIT, "config": {"workload": f"BASELINE.json configs[4] seed {args.sweep_seed}: random LP (m={lp.m}, n={lp.n}, nnz={lp.nnz}), 200 fixed attempts"},
                      "us_per_attempt": us, "algorithmic_bytes": {"k_primal": bp, "k_dual": bd}, "GB/s": (bp + bd) / us / 1e3, "frac_of_peak": (bp + bd) / us / 1e3 / peak}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="UC config index (3 = the 6,049-bus-shaped LP the metric is quoted on)")
    ap.add_argument("--attempts", type=int, default=4096, help="fixed attempts per step (one uc_pdhg_solve_device call)")
    ap.add_argument("--ref-attempts", type=int, default=20)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--clock-sample-ms", type=int, default=100)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--all-configs", action="store_true", help="print the table over all configs instead of the bench line")
    ap.add_argument("--sweep-seed", type=int, default=None, help="run BASELINE.json configs[4] (roofline sweep, seeds 10-14) instead: "
                    "--steps calls of 200 fixed attempts, a short line without e2e (what the ncu DRAM-byte captures of profiles/ run)")
    args = ap.parse_args()
    if args.all_configs:
        return all_configs_table()
    if args.sweep_seed is not None:
        return sweep_line(args)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        return run_reference(args, world, rank)

    import numpy as np
    import torch
    import paper_2607_03627_b200 as P           # fails loudly if the extension is missing; no fallback
    from workloads import uc_config

    assert torch.cuda.is_available(), "bench.py needs a GPU: the product has no CPU path"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    lp = uc_config(args.config)
    h = P.UcLp(lp, device=local_rank)
    info = h.info()
    stream = torch.cuda.Stream(device=dev)
    x = torch.empty(lp.n, dtype=torch.float64, device=dev)
    y = torch.empty(lp.m, dtype=torch.float64, device=dev)
    A = args.attempts

    def step():
        return h.solve_device(x, y, fixed_iterations=A, stream=stream.cuda_stream)

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local_rank, args.clock_sample_ms); sampler.start()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    loop_s = 0.0
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(args.steps):
            s = step()
            launches += s.kernel_launches
            loop_s += s.loop_seconds
        e1.record(stream)
    torch.cuda.synchronize(dev)
    if dist is not None:
        dist.barrier()
    seconds = e0.elapsed_time(e1) * 1e-3
    # dominant kernel, timed live with CUDA events on the launching stream
    primal_ms, dual_ms = h.time_kernels(64, stream=stream.cuda_stream)
    # the same attempts with ONE check at the end instead of one per 64: what the two attempt kernels take inside the
    # graph, under programmatic dependent launch, without the event records that separate them in time_kernels
    nocheck_s = h.solve_device(x, y, fixed_iterations=A, check_every=A, stream=stream.cuda_stream).loop_seconds
    clocks = sampler.stop()
    tmax, units = aggregate(seconds, args.steps * A, dist, dev)

    out = None
    if rank == 0:
        peak, peak_src = load_peaks()
        bp, bd = algorithmic_bytes(lp.m, lp.n, lp.nnz, info)          # what this layout moves (16-bit offsets counted as 2 B)
        sp, sd = algorithmic_bytes(lp.m, lp.n, lp.nnz)                # SURVEY.md 8(d) formula with 32-bit indices everywhere
        dom = ("k_primal", bp, primal_ms) if primal_ms >= dual_ms else ("k_dual", bd, dual_ms)
        ach = dom[1] / (dom[2] * 1e-3) / 1e9
        att_ms = 1e3 * loop_s / (args.steps * A)
        traffic, traffic_src = ncu_traffic(args.config)
        tr = traffic.get(dom[0]) if traffic else None
        ncu_us = traffic.get(dom[0] + "_us_ncu") if traffic else None
        roof = {"bound": "hbm", "kernel": dom[0], "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "what": "frac = effective_frac: ALGORITHMIC bytes of the kernel / its CUDA-event time / the measured copy bandwidth. "
                        "It is NOT the DRAM utilisation: part of the algorithmic bytes (the gathers, the evict_last vectors) is served "
                        "from L2; frac_dram is the same quotient with the DRAM bytes ncu measured.  The ceiling named by \"bound\" is the "
                        "one the byte count is held against; the limiter ncu shows for both attempt kernels is the L2 request rate of "
                        "the 8/16-byte gathers (DESIGN.md section 7), with DRAM at 42-54 % of its peak",
                "effective_frac": ach / peak, "limiter": "l2_requests_of_the_gathers",
                "traffic": tr, "traffic_source": traffic_src if tr else None,
                "frac_dram": (tr / (dom[2] * 1e-3) / 1e9 / peak) if tr else None,
                "kernel_ms_ncu": (ncu_us * 1e-3) if ncu_us else None,
                "kernel_ms_note": "kernel_ms: CUDA events around the kernel with an event record between the two kernels (keeps the next "
                                  "kernel from starting early, so it is an upper bound); kernel_ms_ncu: gpu__time_duration of the same kernel in "
                                  "the committed launch list (cold cache, serialised); in_graph.pair_ms: both kernels inside the graph",
                "peak_source": peak_src, "algorithmic_bytes_per_launch": dom[1], "kernel_ms": dom[2],
                "other_kernel": {"k_primal_ms": primal_ms, "k_dual_ms": dual_ms, "k_primal_bytes": bp, "k_dual_bytes": bd},
                "in_graph": {"what": "context for kernel_ms: an event record between two kernels keeps the next one from starting early "
                                     "(programmatic dependent launch), so the per-kernel event times add up to more than an attempt takes in "
                                     "the graph; pair_ms = both kernels per attempt inside the graph (a run with one check per "
                                     f"{A} attempts), split by the ratio of the event times",
                             "pair_ms": 1e3 * nocheck_s / A, "checks_ms_per_attempt": att_ms - 1e3 * nocheck_s / A,
                             "k_primal_ms_est": 1e3 * nocheck_s / A * primal_ms / (primal_ms + dual_ms),
                             "k_dual_ms_est": 1e3 * nocheck_s / A * dual_ms / (primal_ms + dual_ms)},
                "attempt": {"algorithmic_bytes": bp + bd, "algorithmic_bytes_32bit_indices": sp + sd, "ms_in_graph": att_ms,
                            "GB/s": (bp + bd) / (att_ms * 1e-3) / 1e9,
                            "frac_of_peak": (bp + bd) / (att_ms * 1e-3) / 1e9 / peak,
                            "frac_of_8TBs": (bp + bd) / (att_ms * 1e-3) / 1e9 / 8000.0,
                            "frac_of_8TBs_32bit_formula": (sp + sd) / (att_ms * 1e-3) / 1e9 / 8000.0,
                            "layout_bytes": int(info.bytes_per_attempt)}}
        # ---- e2e: host CSR -> create -> solve to rel KKT 1e-4 -> x, y in host memory
        h2d = lp.row_ptr.nbytes + lp.col_idx.nbytes + lp.val.nbytes + lp.sense.nbytes + lp.b.nbytes + lp.c.nbytes + lp.l.nbytes + lp.u.nbytes
        d2h = 8 * (lp.n + lp.m)
        secs, ttk, its, crs, lps, dts = [], [], [], [], [], []
        for _ in range(max(1, args.e2e_steps)):
            t0 = time.perf_counter()
            h2 = P.UcLp(lp, device=local_rank)
            crs.append(time.perf_counter() - t0)
            s2 = h2.solve()                                  # returns with x, y in host memory
            secs.append(time.perf_counter() - t0)
            t1 = time.perf_counter(); h2.close(); dts.append(time.perf_counter() - t1)
            ttk.append(s2.solve_seconds); its.append(s2.iterations); lps.append(s2.loop_seconds)
            assert s2.status == P.OPTIMAL, P.STATUS_NAMES[s2.status]
        e2e = {"value": its[0] / statistics.median(secs), "unit": UNIT, "job_seconds": secs, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "what": "uc_lp_create(host CSR) + uc_pdhg_solve to rel KKT 1e-4 + x,y to host; attempts / wall seconds of the whole job, "
                       "from the call of uc_lp_create to the return of uc_pdhg_solve (median of the jobs run; every job does the same work)",
               "time_to_kkt_1e-4_s": statistics.median(ttk), "attempts_to_kkt": its[0],
               "create_s": statistics.median(crs), "loop_s": statistics.median(lps), "precondition_s": info.precondition_seconds,
               "first_create_in_process_s": info.create_seconds, "destroy_s_not_in_job": dts}
        out = {"metric": METRIC, "value": units / tmax, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
               "ms_per_step": 1e3 * tmax / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f64", "data": "synthetic",
               "config": {"workload": workload_name(args.config, lp), "attempts_per_step": A, "check_every": 64,
                          "parallelism": "replicas only" if world > 1 else "single GPU", "l2": "inputs_exceed_l2 (working set %.0f MB)" % (info.device_bytes / 1e6)},
               "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof}
        if not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(lp)
    h.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
