"""Re-solves on one handle ("relaxed linear problem", l.62 branch-and-bound): the
matrix, its scalings, both layouts and the captured graph stay on the device; only bounds (uc_lp_update_bounds) or the
objective (uc_lp_update_objective) change, and the next solve may start from the previous point (x0, y0).

    python -m paper_2607_03627_b200.resolve --configs 0 1 2 3

prints, per UC config, the attempts to relative KKT 1e-4 of the sequence  relaxed (cold) -> commitment fixed by
rounding (cold / warm from the relaxed point) -> relaxed again (cold / warm from the fixed point)."""
from __future__ import annotations

import time

from . import binding as _b


def resolve_sequence(lp, fix_commitment, **solve_kwargs):
    """Returns a dict of Solutions: relaxed, fixed_cold, fixed_warm, relaxed_warm (plus wall seconds of each call)."""
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
        pattern = (r.x.reshape(T, V)[:, oU:oU + G].T > 0.5).astype(float)
        fixed = fix_commitment(lp, pattern)
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
    args = ap.parse_args()
    print("| config | relaxed cold: attempts (s) | fixed cold | fixed warm from relaxed | relaxed warm from fixed | objective relaxed / fixed |")
    print("|---|---|---|---|---|---|")
    for c in args.configs:
        lp = uc_config(c)
        o, s = resolve_sequence(lp, fix_commitment)
        cell = lambda k: f"{o[k].iterations} ({s[k]:.3f}){'' if o[k].status == _b.OPTIMAL else ' ' + _b.STATUS_NAMES[o[k].status]}"
        print(f"| {c} | {cell('relaxed')} | {cell('fixed_cold')} | {cell('fixed_warm')} | {cell('relaxed_warm')} | "
              f"{o['relaxed'].primal_obj:.6g} / {o['fixed_warm'].primal_obj:.6g} |", flush=True)


if __name__ == "__main__":
    _main()
