"""N > 1 path of bench.py ("replicas only") on CPU: world_size 2 over gloo.

Each rank steps its own replica; the only collective is the MAX all-reduce of the elapsed time.
"""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1410_4194_b200.driver import aggregate_rate, max_over_ranks


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seconds = 1.0 + rank                      # rank 1 is the slow one
    t = max_over_ranks(seconds, dist)
    rate = aggregate_rate(1000.0, seconds, dist)
    dist.barrier()
    out.put((rank, t, rate))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world2():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, rate in res:
        assert t == 2.0                        # the slowest rank's time on every rank
        assert rate == 2 * 1000.0 / 2.0        # all ranks' units / that time


def test_single_process_is_identity():
    assert max_over_ranks(0.25) == 0.25
    assert aggregate_rate(10.0, 0.5) == 20.0
