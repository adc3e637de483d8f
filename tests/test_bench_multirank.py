"""N > 1 is "replicas only": bench.py sums the units of all ranks and divides by the
MAX over ranks of the timed seconds.  That host logic is covered here with world_size 2 on gloo."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t, u = bench.aggregate(1.0 + rank, 100 * (rank + 1), dist, None)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, t, u))


def test_aggregate_takes_max_time_and_sums_units_over_two_ranks():
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, 2.0, 300.0), (1, 2.0, 300.0)]


def test_aggregate_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(0.5, 7) == (0.5, 7)
    pb, db = bench.algorithmic_bytes(10, 20, 100)
    assert pb + db == 24 * 100 + 76 * 20 + 53 * 10 + 8       # SURVEY.md 8(d) B_iter
