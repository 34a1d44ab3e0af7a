"""World-size-2 gloo test (CPU) of the N>1 host logic: the rank partition of items / pixel tiles covers
everything exactly once, and the max-over-ranks time reduction bench.py uses behaves."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2202_03411_b200.sharding import shard_pixel_tiles, shard_range


def test_shard_range_properties():
    for n in (0, 1, 2, 7, 256, 1000):
        for world in (1, 2, 3, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)
    assert shard_pixel_tiles(1000, 0, 2) == (0, 512) and shard_pixel_tiles(1000, 1, 2) == (512, 1000)


def _worker(rank, world, port, n_items, npix):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_range(n_items, rank, world)
    owned = torch.zeros(n_items, dtype=torch.int64)
    owned[lo:hi] = 1
    dist.all_reduce(owned)                          # every item owned exactly once
    assert bool((owned == 1).all())
    p0, p1 = shard_pixel_tiles(npix, rank, world)
    pix = torch.zeros(npix, dtype=torch.int64)
    pix[p0:p1] = 1
    dist.all_reduce(pix)
    assert bool((pix == 1).all())
    t = torch.tensor([10.0 + rank], dtype=torch.float64)   # max-over-ranks timing as in bench.py
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert t.item() == 10.0 + world - 1
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo_partition():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_worker, args=(2, port, 257, 4097), nprocs=2, join=True)
