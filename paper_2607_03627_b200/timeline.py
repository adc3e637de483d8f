"""Timeline of one PDHG attempt on the device (measurement build).

    python -m paper_2607_03627_b200.timeline [--config 3] [--attempts 24] [--repeats 6]

Builds the library with -DUC_TIMELINE into paper_2607_03627_b200/libuc_pdhg_timeline.so (every warp of k_primal / k_dual
then records %globaltimer marks: kernel entry, grid dependency resolved, own steps done, block sum done, ticket taken,
partials loaded, final sums done, attempt decided), runs `attempts` attempts as plain stream launches under programmatic
dependent launch through uc_pdhg_timeline, and prints where the time of the LAST attempt went, in microseconds from the
moment the first CTA of its k_primal entered.  Needs a GPU.  The product library is not touched."""
from __future__ import annotations

import argparse
import os
import subprocess

import numpy as np

from . import build as _build

TL_LIB = os.path.join(_build.HERE, "libuc_pdhg_timeline.so")


def build_timeline_library() -> str:
    if not os.path.exists(TL_LIB) or any(os.path.getmtime(f) > os.path.getmtime(TL_LIB) for f in _build.DEPENDS):
        subprocess.check_call([_build.nvcc(), *_build.NVCC_FLAGS, "-DUC_TIMELINE", "-o", TL_LIB, *_build.SOURCES])
    return TL_LIB


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--attempts", type=int, default=24)
    ap.add_argument("--repeats", type=int, default=6)
    args = ap.parse_args()
    _build.LIB = build_timeline_library()                   # before the binding loads anything
    from . import binding as B
    from workloads import uc_config
    lp = uc_config(args.config)
    rows, durs = [], {"k_primal": [], "k_dual": []}
    with B.UcLp(lp) as h:
        for _ in range(args.repeats):
            a, b = h.timeline(args.attempts)
            t0 = int(a[:, :, 0][a[:, :, 0] > 0].min())
            rel = lambda v: (np.asarray(v).astype(np.int64) - t0) / 1e3
            rec = {}
            for name, arr in (("k_primal", a), ("k_dual", b)):
                used = arr[:, :, 2] > 0
                nw = int(used.any(0).sum())                                  # warps per CTA incl. the long-row warp
                cons = arr[:, : nw - 1, :]
                ent, dep, done = rel(arr[:, :nw, 0]), rel(cons[:, :, 1]), rel(cons[:, :, 2])
                rec[name] = dict(entry=(ent.min(), ent.max()), dep=(dep.min(), dep.max()),
                                 done=(done.min(), np.median(done), done.max()), exit=rel(arr[:, :nw, 3]).max())
                durs[name].append((cons[:, :, 2].astype(np.int64) - cons[:, :, 1].astype(np.int64)) / 1e3)
            w0 = b[:, 0, :]
            last = int(np.argmax(w0[:, 5]))
            rec["epilogue"] = dict(all_done=rel(b[:, :, 2][b[:, :, 2] > 0]).max(), ticket=rel(w0[last, 4]), loaded=rel(w0[last, 5]),
                                   summed=rel(w0[last, 6]), decided=rel(w0[last, 3]))
            rows.append(rec)
    print(f"# Timeline of one attempt, UC config {args.config} ({lp.m} x {lp.n}, nnz {lp.nnz}); us from the entry of the first k_primal CTA")
    print()
    print("Command: `python -m paper_2607_03627_b200.timeline --config %d --attempts %d --repeats %d` (a -DUC_TIMELINE build of the" % (args.config, args.attempts, args.repeats))
    print("library; plain stream launches with programmatic dependent launch, no events, marks of the last attempt).")
    print()
    print("| repeat | kernel | CTAs enter | dependency resolved | consumer warps done: first / median / last | last exit |")
    print("|---|---|---|---|---|---|")
    for i, r in enumerate(rows):
        for k in ("k_primal", "k_dual"):
            v = r[k]
            print(f"| {i} | {k} | {v['entry'][0]:.1f} .. {v['entry'][1]:.1f} | {v['dep'][0]:.1f} .. {v['dep'][1]:.1f} | "
                  f"{v['done'][0]:.1f} / {v['done'][1]:.1f} / {v['done'][2]:.1f} | {v['exit']:.1f} |")
    print()
    print("| repeat | k_dual epilogue: last warp done | ticket of the last CTA | partials of all CTAs loaded | final sums | attempt decided |")
    print("|---|---|---|---|---|---|")
    for i, r in enumerate(rows):
        e = r["epilogue"]
        print(f"| {i} | {e['all_done']:.2f} | {e['ticket']:.2f} | {e['loaded']:.2f} | {e['summed']:.2f} | {e['decided']:.2f} |")
    print()
    print("| kernel | busy time of a consumer warp (dependency resolved -> own steps done): mean | std over warps and repeats | "
          "std of the per-warp mean (systematic) | mean per-warp std over repeats (random) | max - median |")
    print("|---|---|---|---|---|---|")
    for k, d in durs.items():
        X = np.stack(d)
        print(f"| {k} | {X.mean():.2f} | {X.std():.2f} | {X.mean(0).std():.2f} | {X.std(0).mean():.2f} | "
              f"{np.mean([x.max() - np.median(x) for x in X]):.2f} |")


if __name__ == "__main__":
    main()
