"""uc_lp_spmv_static against uc_lp_spmv (-m gpu).  Collected LAST on purpose (the file name sorts after every other
test file): `pytest -x` stops at the first failure, so a failure here must not hide the parity tests.

Why the entry point exists: uc_lp_spmv allocates four device vectors per call.  Some users of this library cannot
do that -- code that shares the GPU with latency-critical streams (cudaMalloc / cudaFree synchronise the whole device
and stall them), code in a process whose device memory already belongs to a pool or caching allocator (a raw cudaMalloc
then fails), code under a fixed-memory rule after start-up.  For them uc_lp_spmv_static keeps its two intermediate
vectors in a fixed 2 MiB array inside the library, which limits it to handles with m + n <= 262,144 (rounded to 32s).

What is checked: the product is uc_lp_spmv's bit for bit (same kernels, same order of additions), for K~ and for K~',
on two calls in a row with different inputs -- the second call finds the array full of the first call's values and must
not be affected by them -- and again after a call with a smaller LP in between; an LP above the limit is refused with
a message that names the limit.  The test owns the input and output buffers (torch tensors); the entry point only
gets their addresses.  It passes alone in a fresh process and after the rest of the suite: it depends on no state but
the handle it creates, and the first call on the device does the one-time address look-up of the array.
"""
import numpy as np
import pytest

import paper_2607_03627_b200 as P
from paper_2607_03627_b200 import binding
from workloads import tiny, uc_config
from workloads.lp import from_coo

pytestmark = pytest.mark.gpu


def _sparse_lp(seed, m, n, long_rows=0):
    """Seeded LP with 0..8 entries per row, `long_rows` rows beyond the sliced-ELL threshold, three empty rows, sizes as
    given (not multiples of 32 in the callers below)."""
    rng = np.random.default_rng(seed)
    lens = rng.integers(0, 9, m)
    if long_rows:
        lens[rng.integers(3, m, long_rows)] = rng.integers(40, 200, long_rows)
    lens[:3] = 0
    rows = np.repeat(np.arange(m), lens)
    cols = np.concatenate([rng.choice(n, size=int(k), replace=False) for k in lens] + [np.zeros(0, dtype=np.int64)])
    vals = rng.standard_normal(rows.size)
    sense = np.where(rng.uniform(size=m) < 0.5, ord("E"), ord("G")).astype(np.uint8)
    return from_coo(m, n, rows.tolist(), cols.tolist(), vals, sense, np.zeros(m), rng.standard_normal(n),
                    -np.ones(n), np.ones(n), name="no_alloc")


@pytest.mark.parametrize("name", ["uc0", "uc1", "ragged"])
def test_static_scratch_spmv_equals_the_allocating_one_on_consecutive_calls(name):
    import torch
    lp = {"uc0": lambda: uc_config(0), "uc1": lambda: uc_config(1), "ragged": lambda: _sparse_lp(5, 2513, 3007, long_rows=5)}[name]()
    assert (lp.m + 31) // 32 * 32 + (lp.n + 31) // 32 * 32 <= binding.SPMV_STATIC_MAX_DOUBLES
    rng = np.random.default_rng(17)
    with P.UcLp(lp) as h:
        for call in range(2):                                   # two calls in a row, fresh inputs each time
            x = rng.standard_normal(lp.n) * 10.0 ** call
            y = rng.standard_normal(lp.m) * 10.0 ** call
            want_kx, want_kty = h.spmv(x, transpose=False), h.spmv(y, transpose=True)
            dx = torch.from_numpy(x).cuda(); dy = torch.from_numpy(y).cuda()
            okx = torch.full((max(lp.m, 1),), float("nan"), dtype=torch.float64, device="cuda")
            okty = torch.full((max(lp.n, 1),), float("nan"), dtype=torch.float64, device="cuda")
            torch.cuda.synchronize()                            # the handle's stream is not torch's: order by hand
            h.spmv_static(dx.data_ptr(), okx.data_ptr(), transpose=False)
            h.spmv_static(dy.data_ptr(), okty.data_ptr(), transpose=True)      # same stream, right behind: no wait needed
            torch.cuda.synchronize()
            got_kx, got_kty = okx[:lp.m].cpu().numpy(), okty[:lp.n].cpu().numpy()
            np.testing.assert_array_equal(got_kx, want_kx)      # bit for bit: tighter than the 1e-13 the spmv test allows
            np.testing.assert_array_equal(got_kty, want_kty)
            assert np.isfinite(got_kx).all() and np.isfinite(got_kty).all()


def test_static_scratch_keeps_no_state_between_handles():
    """A small LP's call in between leaves its values at the front of the shared array; the larger LP's next call must
    still give the allocating path's result."""
    import torch
    big, small = uc_config(0), tiny.small_random(6, 4, 0)
    rng = np.random.default_rng(23)
    x = rng.standard_normal(big.n); xs = rng.standard_normal(small.n)
    with P.UcLp(big) as hb, P.UcLp(small) as hs:
        want = hb.spmv(x)
        want_s = hs.spmv(xs)
        dx = torch.from_numpy(x).cuda(); dxs = torch.from_numpy(xs).cuda()
        out = torch.empty(big.m, dtype=torch.float64, device="cuda"); outs = torch.empty(small.m, dtype=torch.float64, device="cuda")
        for _ in range(2):
            out.fill_(float("nan")); outs.fill_(float("nan"))
            torch.cuda.synchronize()
            hb.spmv_static(dx.data_ptr(), out.data_ptr())
            torch.cuda.synchronize()                            # two handles = two streams: the calls may not overlap
            hs.spmv_static(dxs.data_ptr(), outs.data_ptr())
            torch.cuda.synchronize()
            hb.spmv_static(dx.data_ptr(), out.data_ptr())
            torch.cuda.synchronize()
            np.testing.assert_array_equal(out.cpu().numpy(), want)
            np.testing.assert_array_equal(outs.cpu().numpy(), want_s)


def test_static_scratch_refuses_an_lp_above_its_limit():
    import torch
    n = binding.SPMV_STATIC_MAX_DOUBLES                          # n alone fills the array; m = 64 more does not fit
    lp = _sparse_lp(3, 64, n)
    with P.UcLp(lp) as h:
        dv = torch.zeros(n, dtype=torch.float64, device="cuda"); out = torch.zeros(64, dtype=torch.float64, device="cuda")
        with pytest.raises(P.UcError) as e:
            h.spmv_static(dv.data_ptr(), out.data_ptr())
        assert e.value.code == -1 and "UC_SPMV_STATIC_MAX_DOUBLES" in str(e.value) and "262144" in str(e.value)
        assert h.spmv(np.zeros(n)).shape == (64,)                # the allocating path still serves it
