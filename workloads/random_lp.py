"""Random bounded sparse LPs for the per-iteration roofline sweep (BASELINE.json configs[4]).

m = n in {1e5, 1e6, 4e6, 1e7, 2e7} with seeds 10..14; nnz/row ~ U{4..12}; nonzeros ~ N(0,1);
bounds [-U(0,10), U(0,10)]; b = A x0 for a random point x0 inside the box; c ~ N(0,1).
Open choices (listed in DESIGN.md): columns ~ U{0..n-1}, sorted, duplicates
dropped; sense 'E' on even rows and 'G' on odd rows.  Data only -- no method arithmetic.
"""
from __future__ import annotations

import numpy as np

from .lp import LP

SWEEP_SIZES = {10: 100_000, 11: 1_000_000, 12: 4_000_000, 13: 10_000_000, 14: 20_000_000}


def sweep_config(seed: int) -> LP:
    return random_lp(SWEEP_SIZES[seed], seed)


def random_lp(n: int, seed: int, m: int | None = None, chunk: int = 2_000_000) -> LP:
    rng = np.random.default_rng(seed)
    m = n if m is None else m
    lens = rng.integers(4, 13, m)
    row_ptr = np.zeros(m + 1, dtype=np.int64)
    cols_out, ptr_counts = [], np.empty(m, dtype=np.int64)
    for s in range(0, m, chunk):                       # chunked so 2e7 rows stay within a few GB
        e = min(m, s + chunk)
        k = lens[s:e]
        cand = rng.integers(0, n, (e - s, 12))
        cand[np.arange(12)[None, :] >= k[:, None]] = n          # sentinel sorts last
        cand.sort(axis=1)
        keep = cand < n
        keep[:, 1:] &= cand[:, 1:] != cand[:, :-1]              # drop duplicates within a row
        ptr_counts[s:e] = keep.sum(axis=1)
        cols_out.append(cand[keep].astype(np.int32))
    np.cumsum(ptr_counts, out=row_ptr[1:])
    col_idx = np.concatenate(cols_out) if cols_out else np.zeros(0, np.int32)
    del cols_out
    nnz = int(row_ptr[-1])
    val = rng.standard_normal(nnz)
    l = -rng.uniform(0.0, 10.0, n)
    u = rng.uniform(0.0, 10.0, n)
    x0 = l + rng.uniform(0.0, 1.0, n) * (u - l)
    c = rng.standard_normal(n)
    # b = A x0 (input construction only): per-row sums of val * x0[col]
    prod = val * x0[col_idx]
    b = np.add.reduceat(prod, row_ptr[:-1]) if nnz else np.zeros(m)
    b[ptr_counts == 0] = 0.0
    sense = np.where(np.arange(m) % 2 == 0, ord("E"), ord("G")).astype(np.uint8)
    return LP(m=m, n=n, row_ptr=row_ptr, col_idx=col_idx, val=val, sense=sense, b=b, c=c, l=l, u=u,
              name=f"random_n{n}_s{seed}", meta=dict(seed=seed, x0=x0))
