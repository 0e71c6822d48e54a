"""N > 1 path of bench.py on CPU: world_size 2, gloo.  Frame pairs are independent,
so ranks take pairs round-robin with no data-path collective; the only communication is the
max-over-ranks reduction of the measured time (replicas only)."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    mine = bench.shard_pairs(11, rank, world)
    t = bench.reduce_max_time(10.0 + 5.0 * rank, dist)
    q.put((rank, mine, t))
    dist.barrier()
    dist.destroy_process_group()


def test_round_robin_shards_and_max_time_over_two_ranks():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0][1] == [0, 2, 4, 6, 8, 10] and got[1][1] == [1, 3, 5, 7, 9]
    assert sorted(got[0][1] + got[1][1]) == list(range(11))        # every pair exactly once
    assert got[0][2] == got[1][2] == 15.0                          # max over ranks on both


def test_single_process_is_identity():
    import bench
    assert bench.shard_pairs(5, 0, 1) == [0, 1, 2, 3, 4]
    assert bench.reduce_max_time(3.5, None) == 3.5
