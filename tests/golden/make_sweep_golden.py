"""Writes tests/golden/oracle_sweep_seed<S>.json: what the CPU oracle (oracle/ only) produces on the roofline-sweep
LPs of BASELINE.json configs[4] after the 200 fixed attempts that `north_star` states, for the sizes where the
oracle needs minutes (seed 12: m = n = 4e6, seed 13: 1e7, seed 14: 2e7).  Calls only oracle/ and workloads/.

The iterates have 4e6 .. 2e7 entries each, so the file stores what a test can compare without them:
  * the full per-attempt trace (200 records: eta_used, eta_bar, eta_next, the three GLOBAL reductions
    |dx|^2, |dy|^2, |dy'K dx| and the accept flag) -- every record is a function of all entries of the iterate;
  * the check trace (k = 64, 128, 192: restart kind, candidate, omega after, mu_c, mu_r, relKKT of both points);
  * |x|_2, |y|_2 and `samples` seeded sample positions of x and y with their values (sampled outputs);
  * four seeded random projections r_q . x and s_q . y (r, s ~ N(0,1), numpy default_rng(777 + q)), which move if
    ANY entry moves.
Usage: python tests/golden/make_sweep_golden.py 12 13 14      (each seed writes its own file; ~3 / 8 / 17 min, 5 / 12 / 25 GB)
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle                         # noqa: E402
from workloads import sweep_config    # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
F = 200
SAMPLES = 2048
PROJECTIONS = 4


def sample_positions(seed, size):
    return np.sort(np.random.default_rng(5000 + seed).choice(size, size=min(SAMPLES, size), replace=False))


def projections(v, which):
    """r_q . v for q = 0..PROJECTIONS-1, r_q ~ N(0,1) from default_rng(777 + 10 q + which), summed with math.fsum-like
    accuracy (numpy pairwise in float64 then longdouble accumulate over chunks)."""
    out = []
    for q in range(PROJECTIONS):
        rng = np.random.default_rng(777 + 10 * q + which)
        acc = np.longdouble(0.0)
        for s in range(0, v.size, 1 << 22):
            r = rng.standard_normal(min(1 << 22, v.size - s))
            acc += np.sum((r * v[s:s + r.size]).astype(np.longdouble))
        out.append(float(acc))
    return out


def main(seeds):
    for seed in seeds:
        t = time.time()
        lp = sweep_config(seed)
        tg = time.time() - t
        t = time.time()
        s = oracle.solve(lp, fixed_iterations=F, trace_attempts=F, trace_checks=64)
        dt = time.time() - t
        ix, iy = sample_positions(seed, lp.n), sample_positions(seed + 100, lp.m)
        a = s.attempts
        data = dict(
            seed=seed, m=lp.m, n=lp.n, nnz=lp.nnz, fixed_iterations=F,
            iterations=int(s.iterations), accepted=int(s.accepted), restarts=int(s.restarts),
            eta=s.eta, omega=s.omega, primal_obj=s.primal_obj, dual_obj=s.dual_obj, rel_kkt=s.rel_kkt,
            attempts=dict(accepted=[int(v) for v in a["accepted"]],
                          **{k: [float(v) for v in a[k]] for k in ("eta_used", "eta_bar", "eta_next", "dx2", "dy2", "inter")}),
            checks=[dict(k=int(c["k"]), restart_kind=int(c["restart_kind"]), candidate=int(c["candidate"]),
                         omega_after=float(c["omega_after"]), mu_c=float(c["mu_c"]), mu_r=float(c["mu_r"]),
                         relkkt_cur=float(c["relkkt_cur"]), relkkt_avg=float(c["relkkt_avg"])) for c in s.checks],
            x_norm=float(np.linalg.norm(s.x)), y_norm=float(np.linalg.norm(s.y)),
            x_pos=[int(v) for v in ix], x_val=[float(v) for v in s.x[ix]],
            y_pos=[int(v) for v in iy], y_val=[float(v) for v in s.y[iy]],
            x_proj=projections(s.x, 0), y_proj=projections(s.y, 1),
            generator_seconds=tg, oracle_seconds=dt, host_cores_used=1)
        out = os.path.join(HERE, f"oracle_sweep_seed{seed}.json")
        with open(out, "w") as f:
            json.dump(data, f, indent=None, separators=(",", ":"), sort_keys=True)
            f.write("\n")
        print(seed, lp.n, f"generator {tg:.0f} s, oracle {dt:.0f} s ({F / dt:.2f} attempts/s)", flush=True)


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [12])
