"""-m "not gpu": the N > 1 path of bench.py is "replicas only": every rank runs
the same step and the only exchange is the max-over-ranks time.  world_size 2 on gloo."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_ms = 2.0 + rank            # rank 1 is the slow one
    ms = bench.replica_max(local_ms, world, "cpu")
    out[rank] = (ms, bench.replica_throughput(3.0e9, ms, world))
    dist.destroy_process_group()


def test_replicas_aggregate_with_slowest_rank():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 3.0                     # max over ranks on both
    assert abs(res[0][1] - 2 * 3.0e9 / 3.0e-3 / 1e9) < 1e-6  # two replicas, slowest time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.replica_max(1.5, 1, "cpu") == 1.5
    assert bench.replica_throughput(1e9, 1.0, 1) == 1000.0
