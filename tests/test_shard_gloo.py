"""N > 1 host logic on CPU: two `gloo` ranks each take their channel shard (paper_1708_00720_b200.shard), run the
oracle on it, and the gathered slabs must equal the single-process result; the max-over-ranks timing reduction
bench.py uses is exercised too.  No GPU and no data-path collective: the gather here is the test's, not the product's."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1708_00720_b200.shard import channel_shard


def test_channel_shard_partitions():
    for nchan in (1, 2, 7, 256, 3072, 16384):
        for world in (1, 2, 3, 8):
            cover = []
            for r in range(world):
                c0, c1 = channel_shard(nchan, world, r)
                assert 0 <= c0 <= c1 <= nchan
                cover.extend(range(c0, c1))
            assert cover == list(range(nchan))
            sizes = [channel_shard(nchan, world, r)[1] - channel_shard(nchan, world, r)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        channel_shard(8, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, C, T, seed, q):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(seed)
        x = rng.integers(0, 256, size=(T, C, 2 * N), dtype=np.uint8)  # ci8 bytes, every rank draws the same span
        c0, c1 = channel_shard(C, world, rank)
        mine = oracle.xcorr(np.ascontiguousarray(x[:, c0:c1]), N, c1 - c0, T, 8)
        # gather the slabs (test plumbing) and take the max over ranks of a fake per-rank time (bench.py's reduction)
        nb = N * (N + 1) // 2
        full = torch.zeros((C, nb, 2), dtype=torch.int32)
        full[c0:c1] = torch.from_numpy(mine)
        dist.all_reduce(full, op=dist.ReduceOp.SUM)
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        # the beamformer shards the same way: span channels and the weight rows of those channels
        K = 3
        w = rng.integers(-127, 128, size=(C, K, 2 * N)).astype(np.int8).view(np.uint8)
        bmine = oracle.beamform(np.ascontiguousarray(x[:, c0:c1]), np.ascontiguousarray(w[c0:c1]), N, c1 - c0, T, K, 8)
        bfull = torch.zeros((T, C, K, 2), dtype=torch.int32)
        bfull[:, c0:c1] = torch.from_numpy(bmine)
        dist.all_reduce(bfull, op=dist.ReduceOp.SUM)
        if rank == 0:
            ref = oracle.xcorr(x, N, C, T, 8)
            bref = oracle.beamform(x, w, N, C, T, K, 8)
            q.put((bool(np.array_equal(full.numpy(), ref)) and bool(np.array_equal(bfull.numpy(), bref)), float(t.item())))
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_and_agree():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, 24, 5, 40, 123, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    same, tmax = q.get()
    assert same
    assert tmax == 11.0
