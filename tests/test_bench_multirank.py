"""N > 1 path of bench.py on CPU (gloo, world_size 2): the path does not shard (DESIGN.md §8,
replicas only), so the only cross-rank logic is the max-over-ranks step time and the whole-job
aggregate; no collective touches the data path."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = 0.070 + 0.010 * rank                 # rank 1 is the slow replica
        slowest = bench.reduce_max_over_ranks(mine, "cpu")
        out[rank] = (slowest, bench.whole_job_value(344_067_072, world, slowest))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value():
    import torch.multiprocessing as mp
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    assert set(out.keys()) == {0, 1}
    for r in range(world):
        slowest, value = out[r]
        assert slowest == pytest.approx(0.080)
        assert value == pytest.approx(2 * 344_067_072 / 0.080e-3 / 1e9)


def test_single_rank_is_identity():
    import bench
    assert bench.reduce_max_over_ranks(0.123) == 0.123
    assert bench.whole_job_value(10**9, 1, 1.0) == pytest.approx(1000.0)
