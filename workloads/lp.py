"""Plain container for one LP in the C-ABI layout (no method arithmetic here)."""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class LP:
    """min c'x  s.t.  (A x)_i = b_i ('E') or >= b_i ('G'),  l <= x <= u.

    CSR: row_ptr int64[m+1], col_idx int32[nnz], val float64[nnz]; sense uint8[m]
    holding ord('E') / ord('G'); absent bounds are -inf / +inf.
    """
    m: int
    n: int
    row_ptr: np.ndarray
    col_idx: np.ndarray
    val: np.ndarray
    sense: np.ndarray
    b: np.ndarray
    c: np.ndarray
    l: np.ndarray
    u: np.ndarray
    name: str = "lp"
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    def validate(self) -> None:
        assert self.row_ptr.dtype == np.int64 and self.row_ptr.shape == (self.m + 1,)
        assert self.col_idx.dtype == np.int32 and self.val.dtype == np.float64
        assert self.col_idx.shape == self.val.shape == (self.nnz,)
        assert self.sense.dtype == np.uint8 and self.sense.shape == (self.m,)
        for v, k in ((self.b, self.m), (self.c, self.n), (self.l, self.n), (self.u, self.n)):
            assert v.dtype == np.float64 and v.shape == (k,)
        assert self.row_ptr[0] == 0 and np.all(np.diff(self.row_ptr) >= 0)
        if self.nnz:
            assert self.col_idx.min() >= 0 and self.col_idx.max() < self.n
        assert np.all(self.l <= self.u)

    def to_scipy(self):
        import scipy.sparse as sp
        return sp.csr_matrix((self.val, self.col_idx, self.row_ptr), shape=(self.m, self.n))

    def dense(self) -> np.ndarray:
        return np.asarray(self.to_scipy().todense())


def from_coo(m, n, rows, cols, vals, sense, b, c, l, u, name="lp", meta=None) -> LP:
    """Assemble an LP from COO triples (sorted by row, then column; no duplicates expected)."""
    rows = np.asarray(rows, dtype=np.int64)
    cols = np.asarray(cols, dtype=np.int64)
    vals = np.asarray(vals, dtype=np.float64)
    order = np.lexsort((cols, rows))
    rows, cols, vals = rows[order], cols[order], vals[order]
    if rows.size > 1:
        dup = (rows[1:] == rows[:-1]) & (cols[1:] == cols[:-1])
        assert not dup.any(), "duplicate (row, col) entry in generator output"
    counts = np.bincount(rows, minlength=m).astype(np.int64)
    row_ptr = np.zeros(m + 1, dtype=np.int64)
    np.cumsum(counts, out=row_ptr[1:])
    lp = LP(m=int(m), n=int(n), row_ptr=row_ptr, col_idx=cols.astype(np.int32), val=vals,
            sense=np.asarray(sense, dtype=np.uint8), b=np.asarray(b, dtype=np.float64),
            c=np.asarray(c, dtype=np.float64), l=np.asarray(l, dtype=np.float64),
            u=np.asarray(u, dtype=np.float64), name=name, meta=meta or {})
    return lp


def from_dense(A, sense, b, c, l, u, name="lp") -> LP:
    A = np.atleast_2d(np.asarray(A, dtype=np.float64))
    m, n = A.shape
    if A.size == 0:
        m = A.shape[0] if A.ndim == 2 else 0
    rows, cols = np.nonzero(A)
    vals = A[rows, cols]
    s = np.frombuffer(("".join(sense)).encode(), dtype=np.uint8) if len(sense) else np.zeros(0, np.uint8)
    return from_coo(m, len(c), rows, cols, vals, s, b, c, l, u, name=name)
