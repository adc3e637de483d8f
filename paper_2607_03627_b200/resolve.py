"""Re-solves on one handle ("relaxed linear problem", l.62 branch-and-bound): the
matrix, its scalings, both layouts and the captured graph stay on the device; only bounds (uc_lp_update_bounds) or the
objective (uc_lp_update_objective) change, and the next solve may start from the previous point (x0, y0).

    python -m paper_2607_03627_b200.resolve --configs 0 1 2 3

prints, per UC config, the attempts to relative KKT 1e-4 of cold and warm re-solves after a branch-and-bound style
fixing, a cost change and a full rounding of the commitment (see resolve_sequence)."""
from __future__ import annotations

import time

from . import binding as _b


def resolve_sequence(lp, fix_commitment, **solve_kwargs):
    """Returns (Solutions, wall seconds) of, all on ONE handle:
        relaxed                      the LP relaxation, cold
        dive_cold / dive_warm        a branch-and-bound style child: every commitment the relaxation left within 1e-3 of
                                     0 or 1 is fixed there (uc_lp_update_bounds); cold, and warm from the relaxed point
        dive_state / cost_state      the same warm starts, carrying the parent's final step size and primal weight too
                                     (uc_pdhg_params.eta0 / omega0, R2b)
        cost_cold / cost_warm        generation costs changed by +-2 % (uc_lp_update_objective), relaxed bounds; cold / warm
        fixed_cold / fixed_warm      the whole commitment fixed by rounding at 0.5 (may be infeasible: ramp and min-up/down
                                     rows do not survive rounding on every instance; PDHG then runs to its iteration limit)
        relaxed_warm                 back to the relaxed bounds and costs, warm from the last point"""
    import numpy as np
    out, sec = {}, {}
    G, T, V, oU = lp.meta["G"], lp.meta["T"], lp.meta["V"], lp.meta["offsets"]["u"]

    def run(h, name, **kw):
        t = time.perf_counter()
        out[name] = h.solve(**solve_kwargs, **kw)
        sec[name] = time.perf_counter() - t

    with _b.UcLp(lp) as h:
        h.solve(fixed_iterations=64)                       # graph instantiation is not part of any timing
        run(h, "relaxed")
        r = out["relaxed"]
        U = r.x.reshape(T, V)[:, oU:oU + G]
        # ---- dive: fix what is (numerically) integral already
        l2 = lp.l.copy().reshape(T, V); u2 = lp.u.copy().reshape(T, V)
        one, zero = U >= 1.0 - 1e-3, U <= 1e-3
        l2[:, oU:oU + G][one] = 1.0; u2[:, oU:oU + G][zero] = 0.0
        out["dive_fixed_share"] = float((one | zero).mean())
        h.update_bounds(l2.ravel(), u2.ravel())
        run(h, "dive_cold")
        run(h, "dive_warm", x0=r.x, y0=r.y)
        run(h, "dive_state", x0=r.x, y0=r.y, eta0=r.eta, omega0=r.omega)
        h.update_bounds(lp.l, lp.u)
        # ---- cost change
        c2 = lp.c * (1.0 + 0.02 * np.sin(np.arange(lp.n) * 0.37))
        h.update_objective(c2)
        run(h, "cost_cold")
        run(h, "cost_warm", x0=r.x, y0=r.y)
        run(h, "cost_state", x0=r.x, y0=r.y, eta0=r.eta, omega0=r.omega)
        h.update_objective(lp.c)
        # ---- the whole commitment rounded
        fixed = fix_commitment(lp, (U.T > 0.5).astype(float))
        h.update_bounds(fixed.l, fixed.u)
        run(h, "fixed_cold")
        run(h, "fixed_warm", x0=r.x, y0=r.y)
        f = out["fixed_warm"]
        h.update_bounds(lp.l, lp.u)
        run(h, "relaxed_warm", x0=f.x, y0=f.y)
    return out, sec


def _main():
    import argparse
    from workloads import fix_commitment, uc_config
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[0, 1, 2])
    ap.add_argument("--iter-limit", type=int, default=100000)
    args = ap.parse_args()
    print("| config | relaxed, cold: attempts (s) | integral commitments fixed (share): cold / warm (x, y) / warm (x, y, eta, omega) | costs +-2 %: cold / warm / warm + state | "
          "whole commitment rounded: cold / warm | relaxed again, warm from the rounded run | objective relaxed / dive / rounded |")
    print("|---|---|---|---|---|---|---|")
    for c in args.configs:
        lp = uc_config(c)
        o, s = resolve_sequence(lp, fix_commitment, iter_limit=args.iter_limit)
        cell = lambda k: f"{o[k].iterations} ({s[k]:.3f}){'' if o[k].status == _b.OPTIMAL else ' ' + _b.STATUS_NAMES[o[k].status]}"
        print(f"| {c} | {cell('relaxed')} | ({o['dive_fixed_share']:.2f}) {cell('dive_cold')} / {cell('dive_warm')} / {cell('dive_state')} | {cell('cost_cold')} / {cell('cost_warm')} / {cell('cost_state')} | "
              f"{cell('fixed_cold')} / {cell('fixed_warm')} | {cell('relaxed_warm')} | "
              f"{o['relaxed'].primal_obj:.6g} / {o['dive_warm'].primal_obj:.6g} / {o['fixed_warm'].primal_obj:.6g} |", flush=True)


if __name__ == "__main__":
    _main()
