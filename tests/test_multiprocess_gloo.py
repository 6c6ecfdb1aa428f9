"""world_size-2 gloo test (CPU) of the only multi-rank logic of this repo: bench.py's max-over-ranks timing and
whole-job aggregation (the path itself is "replicas only": no collective in the data path)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local = [1.0 + rank, 5.0 - 2.0 * rank]           # rank 0: (1, 5); rank 1: (2, 3)
    got = bench.max_over_ranks(local)
    dist.barrier()
    if rank == 0:
        out.put(got)
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [2.0, 5.0]
    sys.path.insert(0, ROOT)
    import bench
    # two replicas of 40,000 particles, 10 steps, slowest rank took 2 s in total
    assert bench.whole_job_value(40000, 10, 2, 2.0) == 400000.0
    assert bench.max_over_ranks([3.5]) == [3.5]      # single process: identity
