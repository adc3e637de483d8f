"""Structure of the synthetic inputs (SURVEY.md 8(d) counts)."""
import numpy as np
import pytest

from workloads import uc_lp, uc_config, UC_CONFIGS, random_lp, fix_commitment

from helpers import highs


def _counts(B, L, G, T, mud):
    n = T * (5 * G + L + 2 * B)
    m = T * (B + L + 3 * G + 1) + 2 * G * (T - 1) + (2 * G * T if mud else 0)
    return m, n


@pytest.mark.parametrize("i", [0, 1, 2])
def test_uc_sizes_match_exact_formulas(i):
    cfg = UC_CONFIGS[i]
    lp = uc_config(i)
    lp.validate()
    m, n = _counts(cfg["B"], cfg["L"], cfg["G"], cfg["T"], cfg["min_updown"])
    assert (lp.m, lp.n) == (m, n)
    B, L, G, T = cfg["B"], cfg["L"], cfg["G"], cfg["T"]
    # nnz without min-up/down: balance G+2L+B, flow 3L, pmin 2G, pmax 3G, logic 3G (+G for t>=1), reserve G, ramps 4G
    base = T * (G + 2 * L + B + 3 * L + 2 * G + 3 * G + 3 * G + G) + (T - 1) * (G + 4 * G)
    if not cfg["min_updown"]:
        assert lp.nnz == base
    else:
        assert base + 2 * G * T * 2 < lp.nnz <= base + 2 * G * T * 7
    lens = np.diff(lp.row_ptr)
    assert (lens == G).sum() >= T                               # the T reserve rows have G entries
    if i >= 1:
        assert lens.max() == G                                  # ... and are the longest rows
    assert set(np.unique(lp.sense)) == {ord("E"), ord("G")}


def test_uc_paper_scale_shape_constants():
    cfg = UC_CONFIGS[3]
    m, n = _counts(cfg["B"], cfg["L"], cfg["G"], cfg["T"], True)
    assert (m, n) == (1_884_800, 2_313_408) and cfg["B"] == 6049       # 6049-bus network


def test_uc_generator_is_deterministic_and_seeded():
    a, b = uc_config(0), uc_config(0)
    for f in ("row_ptr", "col_idx", "val", "b", "c", "l", "u", "sense"):
        np.testing.assert_array_equal(getattr(a, f), getattr(b, f))
    c = uc_lp(**{**UC_CONFIGS[0], "seed": 7})
    assert not np.array_equal(a.val, c.val)


def test_uc_config0_structure_and_feasibility():
    lp = uc_config(0)
    meta = lp.meta
    assert meta["pmax_sum"] == pytest.approx(1.3 * meta["peak_load"], rel=1e-12)
    T, V, B = meta["T"], meta["V"], meta["B"]
    o = meta["offsets"]
    l, u, c = lp.l.reshape(T, V), lp.u.reshape(T, V), lp.c.reshape(T, V)
    assert np.all(l[:, o["theta"]] == 0) and np.all(u[:, o["theta"]] == 0)            # reference bus
    assert np.all(np.isinf(l[:, o["theta"] + 1:o["theta"] + B]))                       # other angles free
    assert np.all(c[:, o["shed"]:o["shed"] + B] == 1e4) and np.all(np.isinf(u[:, o["shed"]:o["shed"] + B]))
    obj, x, _ = highs(lp)
    shed = x.reshape(T, V)[:, o["shed"]:o["shed"] + B].sum()
    assert shed < 0.25 * meta["total_load"]
    f = fix_commitment(lp, np.zeros((meta["G"], T)))
    assert np.all(f.l.reshape(T, V)[:, o["u"]:o["u"] + meta["G"]] == 0)
    assert np.all(f.u.reshape(T, V)[:, o["u"]:o["u"] + meta["G"]] == 0)


def test_random_lp_recipe():
    lp = random_lp(20000, 10)
    lp.validate()
    lens = np.diff(lp.row_ptr)
    assert lens.min() >= 1 and lens.max() <= 12 and 7.5 < lens.mean() < 8.5
    assert np.all(lp.l <= 0) and np.all(lp.u >= 0) and lp.l.min() > -10 and lp.u.max() < 10
    x0 = lp.meta["x0"]
    assert np.all(x0 >= lp.l) and np.all(x0 <= lp.u)
    np.testing.assert_allclose(lp.to_scipy() @ x0, lp.b, rtol=1e-12, atol=1e-12)       # b = A x0: feasible
    assert np.all(lp.sense[0::2] == ord("E")) and np.all(lp.sense[1::2] == ord("G"))
    for i in range(0, 200):                                                             # sorted, no duplicates
        cols = lp.col_idx[lp.row_ptr[i]:lp.row_ptr[i + 1]]
        assert np.all(np.diff(cols) > 0)


def test_tuned_presolve_shape_workload():
    """PAPER.md Table VII (l.241-246): the tuned presolve hands PDHG a 38,238 x 44,822 LP; the named workload has that shape."""
    from workloads import uc_config
    lp = uc_config("tuned_presolve")
    lp.validate()
    assert abs(lp.m - 38238) <= 0.01 * 38238 and abs(lp.n - 44822) <= 0.01 * 44822
    assert lp.name == "uc_tuned_presolve"
