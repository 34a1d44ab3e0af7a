"""Rank -> work partition for multi-GPU runs.

The path has no exchange step: batch items (shapes) are independent and so are detector pixels
(PAPER.md:446-450 splits shapes over workers the same way).  Each rank therefore takes a contiguous,
balanced slice of the items (or of the pixel tiles) and no data-path collective is needed.
"""
from __future__ import annotations

from typing import Tuple


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """[lo, hi) of `n` units owned by `rank`: contiguous, sizes differ by at most one, union = all, disjoint."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_pixel_tiles(npix: int, rank: int, world: int, tile: int = 128) -> Tuple[int, int]:
    """Pixel range [lo, hi) owned by `rank`, aligned to whole 128-pixel tiles of the contraction kernel."""
    ntiles = (npix + tile - 1) // tile
    t0, t1 = shard_range(ntiles, rank, world)
    return min(t0 * tile, npix), min(t1 * tile, npix)
