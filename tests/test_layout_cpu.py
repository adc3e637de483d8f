"""Host logic of ingest step A1 without a GPU: permutations, explicit transpose, SELL-32 layouts and
the static step schedules of the attempt kernels, checked entry by entry against the caller's CSR by the library's
own host-only self-check (include/uc_pdhg.h uc_host_layout_selftest).  What it pins: stored entries are the
caller's, in the caller's order; K' rows come in ascending caller row index (the order of the sequential statement's
column scatter -- bit parity of the row sums depends on it); every slice is scheduled exactly once."""
import numpy as np
import pytest

import paper_2607_03627_b200.binding as B
from workloads import LP, random_lp, tiny, uc_config
from test_gpu_parity import ragged_lp

CASES = {
    "one_by_one": tiny.one_by_one, "two_var": tiny.two_var, "box_rows": lambda: tiny.box_only(with_rows=3),
    "small_random": lambda: tiny.small_random(6, 4, 1), "dispatch": lambda: tiny.economic_dispatch()[0],
    "ragged": ragged_lp, "uc0": lambda: uc_config(0), "uc1": lambda: uc_config(1), "random_2e4": lambda: random_lp(20_000, 21),
}


@pytest.mark.parametrize("name", list(CASES))
def test_layouts_and_schedules_reproduce_the_csr(name):
    B.host_layout_selftest(CASES[name]())


@pytest.mark.parametrize("window,thr,ctas,wpc", [(32, 1, 1, 1), (64, 4, 7, 1), (64, 4, 3, 5), (4096, 32, 1, 15), (100000, 1000, 148, 15),
                                                 (4096, 3, 148, 15), (4096, 32, 296, 7)])
def test_layout_options_and_warp_counts(window, thr, ctas, wpc):
    """Tiny windows, every row long / no row long, more warps (and CTAs) than slices, a single warp."""
    for lp in (ragged_lp(), uc_config(0), uc_config(1)):
        B.host_layout_selftest(lp, sell_window=window, long_row_threshold=thr, sched_ctas=ctas, warps_per_cta=wpc)


def banded_and_wide_lp(n=200_000, m=150_000, seed=4):
    """Rows whose columns lie in a narrow band (16-bit offsets apply) mixed with rows that reach across all 200,000
    columns (slices that stay 32-bit), plus one explicit zero at column 0 (must not be mistaken for padding)."""
    from workloads.lp import from_coo
    rng = np.random.default_rng(seed)
    rows, cols = [], []
    for i in range(m):
        if i % 3000 < 2900:                                        # banded rows
            c = (i * n) // m + rng.choice(2000, size=3, replace=False)
        else:                                                      # wide rows
            c = rng.choice(n, size=4, replace=False)
        c = np.unique(np.clip(c, 0, n - 1))
        rows += [i] * len(c); cols += c.tolist()
    vals = rng.standard_normal(len(rows))
    if cols[0] != 0:
        rows.insert(0, 0); cols.insert(0, 0); vals = np.concatenate([[0.0], vals])
    else:
        vals[0] = 0.0
    return from_coo(m, n, rows, cols, vals, np.full(m, ord("G"), np.uint8), np.zeros(m), rng.standard_normal(n),
                    -np.ones(n), np.ones(n), name="banded_and_wide")


def test_sixteen_bit_column_offsets_on_narrow_and_wide_slices():
    """the self-check decodes every narrow slice back to its 32-bit indices, and checks that a
    slice is wide only when its span does not fit 16 bits -- on an LP that has both kinds."""
    lp = banded_and_wide_lp()
    B.host_layout_selftest(lp)
    B.host_layout_selftest(lp, sell_window=64, long_row_threshold=3)


def test_degenerate_shapes():
    z = np.zeros(0)
    empty = LP(m=0, n=0, row_ptr=np.zeros(1, np.int64), col_idx=np.zeros(0, np.int32), val=z, sense=np.zeros(0, np.uint8),
               b=z, c=z, l=z, u=z)
    B.host_layout_selftest(empty)
    rows_only = LP(m=3, n=0, row_ptr=np.zeros(4, np.int64), col_idx=np.zeros(0, np.int32), val=z,
                   sense=np.full(3, ord("G"), np.uint8), b=np.ones(3), c=z, l=z, u=z)
    B.host_layout_selftest(rows_only)
    B.host_layout_selftest(tiny.box_only())              # columns only


def test_bad_arguments_are_rejected():
    lp = tiny.two_var()
    with pytest.raises(B.UcError):
        B.host_layout_selftest(lp, sell_window=8)
    with pytest.raises(B.UcError):
        B.host_layout_selftest(lp, sched_ctas=0)
    with pytest.raises(B.UcError):
        B.host_layout_selftest(lp, warps_per_cta=0)
