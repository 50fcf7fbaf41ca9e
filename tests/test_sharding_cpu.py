"""World-size-2 CPU test (gloo) of the multi-GPU host logic: channel sharding and the max-over-ranks
throughput aggregation bench.py uses.  The data path itself has no collective."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1702_04728_b200.sharding import job_throughput_gbs, shard_channels, weak_scaling_shard


def test_shard_partition_is_exact():
    for total in (1, 4, 7, 64, 1024):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                first, n = shard_channels(total, world, r)
                got += list(range(first, first + n))
            assert got == list(range(total)), (total, world)
    assert weak_scaling_shard(4, 3) == (12, 4)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    first, n = shard_channels(7, world, rank)
    gathered = [None] * world
    dist.all_gather_object(gathered, (first, n))
    # rank 0 took 3 ms, rank 1 took 5 ms for 1 GB each: job = 2 GB / 5 ms
    gbs, ms = job_throughput_gbs(1e9, 1, 3.0 + 2.0 * rank, dist)
    q.put((rank, gathered, gbs, ms))
    dist.destroy_process_group()


def test_world_size_2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, gathered, gbs, ms in res:
        assert gathered == [(0, 4), (4, 3)]
        assert ms == 5.0 and abs(gbs - 2e9 / 5e-3 / 1e9) < 1e-9
