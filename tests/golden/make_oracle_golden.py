"""Writes tests/golden/oracle_converged.json: what the CPU oracle (oracle/ only) returns on the UC
configs at the default stopping rule (relative KKT <= 1e-4) -- status, attempt count,
restart count, objectives, and wall seconds on this host.  The GPU convergence-parity tests compare
against these stored values for the configs where the oracle takes minutes (1-3); config 0 is re-run
live.  Calls only oracle/ and workloads/.   Usage: python tests/golden/make_oracle_golden.py 1 2 3
"""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle                      # noqa: E402
from workloads import uc_config    # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_converged.json")


def main(configs):
    data = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for i in configs:
        lp = uc_config(i)
        t = time.time()
        s = oracle.solve(lp, trace_checks=4096)
        dt = time.time() - t
        data[f"uc_config{i}"] = dict(
            m=lp.m, n=lp.n, nnz=lp.nnz, status=int(s.status), iterations=int(s.iterations),
            accepted=int(s.accepted), restarts=int(s.restarts), returned_average=int(s.returned_average),
            rel_kkt=s.rel_kkt, primal_obj=s.primal_obj, dual_obj=s.dual_obj, omega=s.omega, eta=s.eta,
            restart_trace=[[int(c["k"]), int(c["restart_kind"]), int(c["candidate"])] for c in s.checks if c["restart_kind"]],
            oracle_seconds=dt, host_cores_used=1)
        json.dump(data, open(OUT, "w"), indent=1, sort_keys=True)
        print(i, data[f"uc_config{i}"]["iterations"], dt, flush=True)


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [0, 1, 2])
