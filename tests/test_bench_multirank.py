"""The N > 1 path of bench.py is 'replicas only': no data-path collective, only the
barrier / max-over-ranks timing reduction.  That reduction is exercised here with two gloo ranks on the CPU."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dist.barrier()
        t = bench.max_over_ranks(1.0 + rank, dist, "cpu")          # rank r took 1 + r seconds
        v = bench.replica_throughput(100.0, 3, world, t)
        with open(os.path.join(out, "r%d.txt" % rank), "w") as f:
            f.write("%r %r" % (t, v))
    finally:
        dist.destroy_process_group()


def test_two_rank_timing_reduction(tmp_path):
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        t, v = map(float, open(tmp_path / ("r%d.txt" % r)).read().split())
        assert t == 2.0                       # the slowest rank's time, on every rank
        assert v == pytest.approx(2 * 100.0 * 3 / 2.0)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(0.25) == 0.25
    assert bench.replica_throughput(10.0, 4, 1, 2.0) == 20.0
