"""World-size-2 gloo test (CPU) of the N>1 host logic: the rank partition of items / pixel tiles covers
everything exactly once, and the max-over-ranks time reduction bench.py uses behaves."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import numpy as np

from oracle import oracle as O
from paper_2202_03411_b200.sharding import shard_detector_rows, shard_range


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


def test_row_bands_tile_the_detector_and_reproduce_its_qmap_exactly():
    """Pixel sharding: the q-maps of the row bands (each a detector with its own npy and cy), concatenated, ARE the q-map of the
    full detector -- bit for bit, so a band simulates exactly the pixels it replaces (oracle q-map, Eq. 3)."""
    for (npx, npy, th, lam, cx, cy) in [(64, 64, 30.0, 20.0, 0.0, 0.0), (37, 21, 60.0, 10.0, 1.5, -2.0), (16, 5, 45.0, 3.0, 0.0, 0.5)]:
        full = O.qmap(npx, npy, th, lam, cx, cy)
        for world in (1, 2, 3, 8):
            parts, rows = [], 0
            for r in range(world):
                y0, y1, cyb = shard_detector_rows(npy, cy, r, world)
                assert y0 == rows
                rows = y1
                if y1 > y0:
                    parts.append(O.qmap(npx, y1 - y0, th, lam, cx, cyb))
            assert rows == npy
            assert np.array_equal(np.concatenate(parts), full)


def _worker(rank, world, port, n_items, npix):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_range(n_items, rank, world)
    owned = torch.zeros(n_items, dtype=torch.int64)
    owned[lo:hi] = 1
    dist.all_reduce(owned)                          # every item owned exactly once
    assert bool((owned == 1).all())
    # pixel sharding as bench.py --shard pixels does it: every rank fills its row band, rank 0 gathers the padded bands
    npx, npy = 8, npix
    y0, y1, _ = shard_detector_rows(npy, 0.0, rank, world)
    rows_max = (npy + world - 1) // world
    band = torch.zeros((rows_max, npx), dtype=torch.float32)
    band[: y1 - y0] = (torch.arange(y0, y1, dtype=torch.float32)[:, None] * npx + torch.arange(npx, dtype=torch.float32)[None, :])
    got = [torch.empty_like(band) for _ in range(world)] if rank == 0 else None
    dist.gather(band, got, dst=0)
    if rank == 0:
        full = torch.cat([got[r][: shard_range(npy, r, world)[1] - shard_range(npy, r, world)[0]] for r in range(world)])
        assert torch.equal(full, torch.arange(npy * npx, dtype=torch.float32).reshape(npy, npx))
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
    mp.spawn(_worker, args=(2, port, 257, 41), nprocs=2, join=True)
