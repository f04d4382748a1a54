"""N > 1 bookkeeping of bench.py on CPU (gloo, world_size 2): the path does not shard inside a
problem (replicas only, no data-path collective), so the only multi-rank
logic is the max-over-ranks of the device times and the whole-job rate built from it."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times = [1.0 + rank, 5.0 - rank, 2.0]          # rank 1 slowest in [0], rank 0 in [1]
    got = bench.max_over_ranks(times, dist, torch.device("cpu"))
    dist.barrier()
    out[rank] = got
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_world_size_2():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    assert out[0] == out[1] == [2.0, 5.0, 2.0]
    sys.path.insert(0, ROOT)
    import bench
    # weak scaling over replicas: both ranks' units over the slowest rank's time
    assert bench.whole_job_rate(100.0, world, 2.0) == 100.0
    assert bench.max_over_ranks([3.0], None, torch.device("cpu")) == [3.0]
