"""Beam-major exchange, host logic on CPU (gloo, world size 2): the all-to-all re-layout of
paper_1702_04728_b200/beam_major.py turns channel-sharded beams into beam-sharded ones."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1702_04728_b200 import beam_major


def test_beam_shard_partitions_all_beams():
    for world in (1, 2, 4, 8, 64):
        got = [beam_major.beam_shard(world, r) for r in range(world)]
        assert got[0][0] == 0 and sum(n for _, n in got) == 1024
        assert all(got[r][0] + got[r][1] == got[r + 1][0] for r in range(world - 1))
    with pytest.raises(ValueError):
        beam_major.beam_shard(3, 0)
    assert beam_major.receive_shape(8, 5, 4) == (8, 5, 256, 16)


def _full(C_total, R):
    rng = np.random.default_rng(5)
    return rng.integers(0, 256, size=(C_total, R, 1024, 16), dtype=np.uint8)


def _worker(rank, world, port, C_local, R, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    full = _full(world * C_local, R)
    local = torch.from_numpy(full[rank * C_local:(rank + 1) * C_local].copy())
    recv = beam_major.exchange_all_to_all(local).numpy()
    b0, nb = beam_major.beam_shard(world, rank)
    ok = recv.shape == beam_major.receive_shape(world * C_local, R, world) and np.array_equal(recv, full[:, :, b0:b0 + nb])
    q.put((rank, bool(ok)))
    dist.destroy_process_group()


def test_all_to_all_relayout_world2():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, 3, 4, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
    assert res == [(0, True), (1, True)]


def test_single_rank_is_a_plain_view():
    full = _full(2, 3)
    recv = beam_major.exchange_all_to_all(torch.from_numpy(full)).numpy()
    assert np.array_equal(recv, full)
