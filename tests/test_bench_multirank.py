"""The N > 1 path of bench.py is "replicas only": every rank solves its own
copy and the ranks only exchange bookkeeping.  That bookkeeping is covered here with two gloo
ranks on the CPU."""
import os
import sys

import pytest

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    iters = 217 * (rank + 1)                 # rank 0: 217 iterations, rank 1: 434
    secs = 0.003 * (2 - rank)                # rank 0 is the slow one: 6 ms against 3 ms
    value, n, t = bench.whole_job_value(dist, "cpu", iters, secs)
    mx = bench.reduce_over_ranks(dist, float(rank), "max", "cpu")
    out[rank] = (value, n, t, mx)
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_value_over_two_gloo_ranks():
    import torch.multiprocessing as mp
    mgr = mp.Manager()
    out = mgr.dict()
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert set(out.keys()) == {0, 1}
    for r in (0, 1):
        value, n, t, mx = out[r]
        assert n == 217 + 434 and abs(t - 0.006) < 1e-12 and mx == 1.0
        assert abs(value - 651 / 0.006) < 1e-6
    assert out[0] == out[1]


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(None, "cpu", 100, 0.5) == (200.0, 100.0, 0.5)
