"""The N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- every rank
times its own replica, the job time is the maximum over ranks, the value is the sum of the replicas' work."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = 2.0 + 3.0 * rank                     # ms per K steps measured by this rank
    slowest = bench.max_over_ranks(mine, dist, "cpu")
    value = bench.aggregate_throughput(1000, 4, slowest, world)
    dist.barrier()
    out.put((rank, slowest, value))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_two_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slowest, value in res:
        assert slowest == 5.0                                  # the slower replica sets the job time
        assert abs(value - 2 * 1000 * 4 / 5.0e-3) < 1e-6       # both replicas' work over that time


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.25, None) == 1.25
