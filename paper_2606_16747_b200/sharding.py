"""Multi-GPU sharding of one frame: every pixel and every 64x64 tile is
independent, so a frame splits into contiguous pixel-row bands with NO data-path collective.
Band boundaries are multiples of 64 rows (whole quadtree tiles) chosen so that each rank gets
about F / world_size fragments (balance by fragments, not pixels).  Host logic only: numpy
index arithmetic on `offsets`; no arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np

TILE = 64


def shard_rows(offsets: np.ndarray, width: int, height: int, world_size: int) -> list:
    """Row bands [(y0, y1)] * world_size, 64-row aligned, fragment-balanced, covering [0, H).

    A band may be empty (y0 == y1) when there are fewer 64-row strips than ranks."""
    strips = -(-height // TILE)
    # fragments before each strip boundary
    ys = np.minimum(np.arange(strips + 1) * TILE, height)
    cum = offsets[ys.astype(np.int64) * width].astype(np.int64)
    total = int(cum[-1])
    bounds = [0]
    for r in range(1, world_size):
        target = total * r / world_size
        k = int(np.searchsorted(cum, target, side="left"))
        # nearest strip boundary to the ideal split, monotone
        if k > 0 and k <= strips and abs(cum[k - 1] - target) <= abs(cum[min(k, strips)] - target):
            k -= 1
        k = min(max(k, bounds[-1]), strips)
        bounds.append(k)
    bounds.append(strips)
    return [(int(ys[a]), int(ys[b])) for a, b in zip(bounds[:-1], bounds[1:])]


def slice_rows(offsets: np.ndarray, depth: np.ndarray, rgba: np.ndarray, width: int, y0: int, y1: int):
    """Rebased CSR arrays of rows [y0, y1): (offsets', depth', rgba')."""
    p0, p1 = y0 * width, y1 * width
    f0, f1 = int(offsets[p0]), int(offsets[p1])
    off = (offsets[p0:p1 + 1].astype(np.int64) - f0).astype(np.uint32)
    return off, depth[f0:f1], rgba[f0:f1]


def gather_rows(parts: list, bands: list, width: int, height: int, channels: int) -> np.ndarray:
    """Reassemble per-band outputs ([rows*W, channels] each) into the full [H*W, channels] image."""
    shape = (height * width, channels) if channels > 1 else (height * width,)
    out = np.zeros(shape, parts[0].dtype)
    for part, (y0, y1) in zip(parts, bands):
        out[y0 * width:y1 * width] = part.reshape((-1, channels) if channels > 1 else (-1,))
    return out
