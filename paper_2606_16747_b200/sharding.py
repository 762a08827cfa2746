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


# ---- reprojection across bands (S8): a row halo of the previous frame ----------------------
def halo_rows(height: int, max_motion: float = 0.02) -> int:
    """Rows of `prev_trans` / `prev_depth` a band needs from each neighbour so that every source
    pixel of a reprojection with at most `max_motion` * H of vertical screen motion is local
    (ceil(0.02 H) + 1; BASELINE.json cfg5: <= 2 % screen motion per frame)."""
    return int(np.ceil(max_motion * height)) + 1


def extended_band(band, halo: int, height: int):
    """[y0 - halo, y1 + halo) clipped to the frame."""
    y0, y1 = band
    return max(0, y0 - halo), min(height, y1 + halo)


def band_matrix(M: np.ndarray, height: int, y0: int, y1: int) -> np.ndarray:
    """Reprojection matrix of the rows [y0, y1) seen as a frame of their own.

    noit_reproject works in the NDC of the buffer it is given (pixel centre y + 0.5 over the
    buffer's height, y down, A23).  A band's NDC is an affine image of the frame's:
    y_frame = s * y_band + t with s = (y1 - y0) / H, t = s + 2 y0 / H - 1.  So the band's matrix is
    G2L . M . L2G (float64 here, cast by the caller), both current and previous buffers being the
    same rows.  Coordinate bookkeeping only: the transform itself runs in the kernel."""
    s = (y1 - y0) / height
    t = s + 2.0 * y0 / height - 1.0
    l2g = np.eye(4)
    l2g[1, 1], l2g[1, 3] = s, t
    g2l = np.eye(4)
    g2l[1, 1], g2l[1, 3] = 1.0 / s, -t / s
    return g2l @ np.asarray(M, np.float64) @ l2g


def exchange_halo_rows(band_rows, halo: int, rank: int, world_size: int, group=None):
    """Send this rank's first / last `halo` rows to the neighbouring ranks and receive theirs.

    `band_rows` is a torch tensor [rows, ...] (prev_trans or prev_depth of this rank's band).
    Returns (above, below): the neighbour rows that precede / follow the band (None at the frame
    edge).  One send + one receive per neighbour (`torch.distributed` P2P: NCCL moves them over
    NVLink peer to peer, gloo on the CPU); bands shorter than `halo` rows send what they have.
    The only data-path exchange of the sharded path, and only reprojection needs it."""
    import torch
    import torch.distributed as dist
    ops, above, below = [], None, None
    n = band_rows.shape[0]
    h = min(halo, n)
    counts = [torch.zeros(1, dtype=torch.int64, device=band_rows.device) for _ in range(2)]
    # neighbours' band heights may be below `halo`: exchange the row counts first
    mine = torch.tensor([h], dtype=torch.int64, device=band_rows.device)
    if rank > 0:
        ops += [dist.P2POp(dist.isend, mine, rank - 1, group), dist.P2POp(dist.irecv, counts[0], rank - 1, group)]
    if rank < world_size - 1:
        ops += [dist.P2POp(dist.isend, mine, rank + 1, group), dist.P2POp(dist.irecv, counts[1], rank + 1, group)]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    ops = []
    if rank > 0:
        above = torch.empty((int(counts[0].item()),) + tuple(band_rows.shape[1:]), dtype=band_rows.dtype,
                            device=band_rows.device)
        ops += [dist.P2POp(dist.isend, band_rows[:h].contiguous(), rank - 1, group),
                dist.P2POp(dist.irecv, above, rank - 1, group)]
    if rank < world_size - 1:
        below = torch.empty((int(counts[1].item()),) + tuple(band_rows.shape[1:]), dtype=band_rows.dtype,
                            device=band_rows.device)
        ops += [dist.P2POp(dist.isend, band_rows[n - h:].contiguous(), rank + 1, group),
                dist.P2POp(dist.irecv, below, rank + 1, group)]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    return above, below


# ---- 2:1 tile balance across bands (NEXT-1): a halo of ORIGINAL masks ------------------------
def balance_band(ctx, band_mask, width: int, y0: int, y1: int, frame_height: int, above=None, below=None,
                 iterations: int = 2, delta2: float = 2.2, delta3: float = 3.0):
    """2:1 balance of one band so that the result equals the whole-frame balance bit for bit.

    k Jacobi steps read ORIGINAL masks within Manhattan distance k, so a band needs
    its neighbours' nearest k tile rows of original masks ("a 1-tile halo per
    iteration"): `above` / `below` are those rows ([rows * Tx] int32 tensors, e.g. from
    exchange_halo_rows on the masks viewed as [tile rows, Tx]; None at the frame edge).  The band is
    balanced inside the extended strip, then cell levels, histogram and tile levels of its OWN tiles
    are recomputed with an iterations = 0 call.  Marshalling only: both steps run in balance_kernel.
    Returns noit.quadtree_balance's dict for the band (the `scales` in it are band-local: the
    frame's demand index needs the sum of the bands' histograms)."""
    import torch
    Tx = (width + TILE - 1) // TILE
    ra = 0 if above is None else above.numel() // Tx
    rb = 0 if below is None else below.numel() // Tx
    parts = [t for t in (above, band_mask, below) if t is not None]
    ext = torch.cat([p.reshape(-1) for p in parts]).contiguous()
    ya, yb = y0 - TILE * ra, min(frame_height, y1 + TILE * rb)
    ctx.quadtree_balance(ext, width, yb - ya, iterations=iterations, delta2=delta2, delta3=delta3)
    own = ext[ra * Tx: ra * Tx + band_mask.numel()].clone()
    return ctx.quadtree_balance(own, width, y1 - y0, iterations=0, delta2=delta2, delta3=delta3)
