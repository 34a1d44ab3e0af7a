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


def shard_detector_rows(npy: int, cy: float, rank: int, world: int) -> Tuple[int, int, float]:
    """Pixel sharding ("partition pixel tiles across GPUs, each GPU writes its slice of I"): rank `rank` of `world`
    simulates the rows [y0, y1) of the flat detector.  A row band IS a detector of the C ABI: same npx, theta_max_deg and cx
    (the pixel pitch depends on npx only), npy = y1 - y0 rows and the centre offset cy_band returned here, which puts band row
    iy at the v of full-detector row y0 + iy:  (iy + 1/2 - (y1-y0)/2 + cy_band) = (y0 + iy + 1/2 - npy/2 + cy).
    Returns (y0, y1, cy_band); bands are contiguous, balanced, disjoint and cover every row."""
    y0, y1 = shard_range(npy, rank, world)
    return y0, y1, float(y0) - 0.5 * float(npy) + 0.5 * float(y1 - y0) + float(cy)
