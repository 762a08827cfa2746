"""Seeded procedural rasteriser: screen-space primitives -> per-pixel CSR fragment buffer.

This module is INPUT GENERATION ONLY.  It stands in for the paper's three raster geometry
passes (PAPER.md:55 §3, :95 §3.3), which need a graphics API that does not exist on this box.
It holds none of the method's arithmetic (no selection, no tail reduction, no MLP, no
compositing, no quadtree, no reprojection); both the CPU oracle and the CUDA path are fed the
arrays it returns, byte for byte.

Layout produced:
  offsets u32[P+1]  row-major pixels p = y*W + x, offsets[0] = 0, non-decreasing
  depth   f32[F]    smaller = nearer, in (0, 1)
  rgba    f16[F,4] or f32[F,4]  straight (non-premultiplied) colour, .w = alpha
Fragments of a pixel are contiguous and in SUBMISSION order (primitive id), not depth order.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

KIND_RECT = 0      # geom = (cx, cy, hx, hy, -, -, -, -)           |px-cx|<=hx and |py-cy|<=hy
KIND_ELLIPSE = 1   # geom = (cx, cy, a, b, cos t, sin t, -, -)     (u/a)^2 + (v/b)^2 <= 1
KIND_QUAD = 2      # edges[4,3]: e_k = A*px + B*py + C >= 0 for all k (convex quad)

REGION_ALL = 0     # primitive drawn everywhere
REGION_DETAIL = 1  # only in tiles NOT flagged smooth
REGION_SMOOTH = 2  # only in tiles flagged smooth


@dataclass
class Primitives:
    """Struct-of-arrays list of screen-space primitives, in submission order.

    All coordinates are FULL-RESOLUTION pixel units (pixel (x, y) has its centre at
    (x + 0.5, y + 0.5)).  Depth and colour are affine in screen space:
      z(px, py)   = zplane[i] . (1, px, py)          clipped to [1e-3, 1 - 1e-3]
      c_k(px, py) = cplane[i, k] . (1, px, py)       clipped to [0, 1],  k = r, g, b
    """
    kind: np.ndarray      # int32 [n]
    geom: np.ndarray      # float64 [n, 8]
    edges: np.ndarray     # float64 [n, 4, 3] (KIND_QUAD only)
    bbox: np.ndarray      # float64 [n, 4] = (xmin, ymin, xmax, ymax) in pixel units
    zplane: np.ndarray    # float64 [n, 3]
    cplane: np.ndarray    # float64 [n, 3, 3]
    alpha: np.ndarray     # float64 [n]
    region: np.ndarray    # int32 [n]

    def __len__(self) -> int:
        return int(self.kind.shape[0])

    @staticmethod
    def empty(n: int) -> "Primitives":
        return Primitives(
            kind=np.zeros(n, np.int32), geom=np.zeros((n, 8)), edges=np.zeros((n, 4, 3)),
            bbox=np.zeros((n, 4)), zplane=np.zeros((n, 3)), cplane=np.zeros((n, 3, 3)),
            alpha=np.zeros(n), region=np.zeros(n, np.int32))

    def scaled(self, s: float) -> "Primitives":
        """Same primitives with rect/ellipse extents multiplied by s about their centres."""
        out = Primitives(self.kind.copy(), self.geom.copy(), self.edges.copy(), self.bbox.copy(),
                         self.zplane.copy(), self.cplane.copy(), self.alpha.copy(),
                         self.region.copy())
        m = out.kind != KIND_QUAD
        out.geom[m, 2:4] *= s
        out.update_bbox()
        return out

    def update_bbox(self) -> None:
        for i in range(len(self)):
            k = self.kind[i]
            g = self.geom[i]
            if k == KIND_RECT:
                self.bbox[i] = (g[0] - g[2], g[1] - g[3], g[0] + g[2], g[1] + g[3])
            elif k == KIND_ELLIPSE:
                ex = np.hypot(g[2] * g[4], g[3] * g[5])
                ey = np.hypot(g[2] * g[5], g[3] * g[4])
                self.bbox[i] = (g[0] - ex, g[1] - ey, g[0] + ex, g[1] + ey)
            # KIND_QUAD: bbox is set by the creator from the projected vertices


@dataclass
class FragBuf:
    """Host-side CSR fragment buffer."""
    width: int
    height: int
    offsets: np.ndarray   # uint32 [P+1]
    depth: np.ndarray     # float32 [F]
    rgba: np.ndarray      # float16 or float32 [F, 4]
    meta: dict = field(default_factory=dict)

    @property
    def num_pixels(self) -> int:
        return self.width * self.height

    @property
    def num_fragments(self) -> int:
        return int(self.offsets[-1])

    @property
    def color_fmt(self) -> int:
        return 0 if self.rgba.dtype == np.float16 else 1

    def counts(self) -> np.ndarray:
        return np.diff(self.offsets.astype(np.int64)).astype(np.uint32)

    def rows(self, y0: int, y1: int) -> "FragBuf":
        """Rebased sub-buffer of pixel rows [y0, y1) (used for sampling and for sharding)."""
        p0, p1 = y0 * self.width, y1 * self.width
        f0, f1 = int(self.offsets[p0]), int(self.offsets[p1])
        off = (self.offsets[p0:p1 + 1].astype(np.int64) - f0).astype(np.uint32)
        return FragBuf(self.width, y1 - y0, off, self.depth[f0:f1].copy(),
                       self.rgba[f0:f1].copy(), dict(self.meta))


def _coverage(prims: Primitives, i: int, px: np.ndarray, py: np.ndarray) -> np.ndarray:
    """Boolean inside test for primitive i at sample positions (px[None,:], py[:,None])."""
    k = prims.kind[i]
    g = prims.geom[i]
    X = px[None, :]
    Y = py[:, None]
    if k == KIND_RECT:
        return (np.abs(X - g[0]) <= g[2]) & (np.abs(Y - g[1]) <= g[3])
    if k == KIND_ELLIPSE:
        dx = X - g[0]
        dy = Y - g[1]
        u = (dx * g[4] + dy * g[5]) / g[2]
        v = (-dx * g[5] + dy * g[4]) / g[3]
        return (u * u + v * v) <= 1.0
    e = prims.edges[i]
    m = (e[0, 0] * X + e[0, 1] * Y + e[0, 2]) >= 0.0
    for j in range(1, 4):
        m &= (e[j, 0] * X + e[j, 1] * Y + e[j, 2]) >= 0.0
    return m


def _sample_window(prims: Primitives, i: int, Wr: int, Hr: int, r: int):
    """Index window [x0,x1) x [y0,y1) of r-res pixels whose centres can be inside bbox i."""
    xmin, ymin, xmax, ymax = prims.bbox[i]
    # sample centre of r-res pixel X is (X + 0.5) * r
    x0 = max(int(np.floor(xmin / r - 0.5)), 0)
    y0 = max(int(np.floor(ymin / r - 0.5)), 0)
    x1 = min(int(np.ceil(xmax / r + 0.5)) + 1, Wr)
    y1 = min(int(np.ceil(ymax / r + 0.5)) + 1, Hr)
    return x0, y0, x1, y1


def _covered_pixels(prims: Primitives, i: int, Wr: int, Hr: int, r: int,
                    smooth_tiles: np.ndarray | None, tile: int):
    """Flat r-res pixel ids covered by primitive i, plus their sample positions (full-res units)."""
    x0, y0, x1, y1 = _sample_window(prims, i, Wr, Hr, r)
    if x1 <= x0 or y1 <= y0:
        z = np.zeros(0, np.int64)
        return z, np.zeros(0), np.zeros(0)
    px = (np.arange(x0, x1, dtype=np.float64) + 0.5) * r
    py = (np.arange(y0, y1, dtype=np.float64) + 0.5) * r
    m = _coverage(prims, i, px, py)
    reg = prims.region[i]
    if reg != REGION_ALL and smooth_tiles is not None:
        tx = np.minimum((px // tile).astype(np.int64), smooth_tiles.shape[1] - 1)
        ty = np.minimum((py // tile).astype(np.int64), smooth_tiles.shape[0] - 1)
        sm = smooth_tiles[ty[:, None], tx[None, :]]
        m &= sm if reg == REGION_SMOOTH else ~sm
    yy, xx = np.nonzero(m)
    pix = (yy + y0).astype(np.int64) * Wr + (xx + x0)
    return pix, px[xx], py[yy]


def count_fragments(prims: Primitives, width: int, height: int, r: int = 1, cap: int = 1 << 30,
                    smooth_tiles: np.ndarray | None = None, tile: int = 64) -> np.ndarray:
    """Per-pixel fragment counts (capped) of the r-res raster; used for size calibration."""
    Wr, Hr = -(-width // r), -(-height // r)
    counts = np.zeros(Wr * Hr, np.int32)
    for i in range(len(prims)):
        pix, _, _ = _covered_pixels(prims, i, Wr, Hr, r, smooth_tiles, tile)
        if pix.size:
            keep = counts[pix] < cap
            counts[pix[keep]] += 1
    return counts


def rasterize(prims: Primitives, width: int, height: int, r: int = 1, cap: int = 1 << 30,
              color_dtype=np.float16, smooth_tiles: np.ndarray | None = None,
              tile: int = 64) -> FragBuf:
    """Rasterise `prims` at 1/r resolution (r in {1,2,4}) into a CSR fragment buffer.

    The r-res image is ceil(W/r) x ceil(H/r); r-res pixel (X, Y) samples the primitives at the
    full-res position ((X+0.5)*r, (Y+0.5)*r).  Fragments beyond the
    `cap`-th of a pixel are dropped in submission order.  Colours (and alpha) are rounded to
    `color_dtype` here, before either implementation sees them.
    """
    Wr, Hr = -(-width // r), -(-height // r)
    P = Wr * Hr
    counts = np.zeros(P, np.int32)
    kept = []
    for i in range(len(prims)):
        pix, sx, sy = _covered_pixels(prims, i, Wr, Hr, r, smooth_tiles, tile)
        if pix.size:
            keep = counts[pix] < cap
            if not keep.all():
                pix, sx, sy = pix[keep], sx[keep], sy[keep]
            counts[pix] += 1
        kept.append((pix, sx, sy))
    offsets64 = np.zeros(P + 1, np.int64)
    np.cumsum(counts, out=offsets64[1:])
    F = int(offsets64[-1])
    if F >= 2 ** 32 or P + 1 >= 2 ** 32:
        raise ValueError("fragment buffer exceeds u32 indexing")
    depth = np.empty(F, np.float32)
    rgba = np.empty((F, 4), color_dtype)
    cursor = offsets64[:-1].copy()
    for i, (pix, sx, sy) in enumerate(kept):
        if not pix.size:
            continue
        pos = cursor[pix]
        cursor[pix] += 1
        zp = prims.zplane[i]
        z = np.clip(zp[0] + zp[1] * sx + zp[2] * sy, 1e-3, 1.0 - 1e-3)
        depth[pos] = z.astype(np.float32)
        cp = prims.cplane[i]
        for k in range(3):
            c = np.clip(cp[k, 0] + cp[k, 1] * sx + cp[k, 2] * sy, 0.0, 1.0)
            rgba[pos, k] = c.astype(color_dtype)
        rgba[pos, 3] = color_dtype(prims.alpha[i])
    return FragBuf(Wr, Hr, offsets64.astype(np.uint32), depth, rgba)


def inject_front_ties(fb: FragBuf, rng: np.random.Generator, fraction: float,
                      pixel_mask: np.ndarray | None = None) -> int:
    """Give ~`fraction` of the pixels with n_p >= 2 an exact depth tie AT THE FRONT.

    `pixel_mask` (bool [P], optional) restricts the eligible pixels (cfg4: detail tiles only --
    a tie reorders the layers of a pixel, which in a smooth region is salt-and-pepper noise).

    In each chosen pixel the bit pattern of the minimum depth is copied onto one other,
    uniformly chosen fragment of that pixel, so the tie sits on either side of the index order
    (BASELINE.json cfg3: "10% of pixels have exact depth ties").  Returns the number of pixels
    modified.  Pure input manipulation.
    """
    off = fb.offsets.astype(np.int64)
    n = np.diff(off)
    P = n.shape[0]
    cand = np.nonzero((n >= 2) if pixel_mask is None else ((n >= 2) & pixel_mask))[0]
    if cand.size == 0:
        return 0
    chosen = cand[rng.random(cand.size) < fraction]
    if chosen.size == 0:
        return 0
    starts = off[:-1]
    nonempty = np.nonzero(n > 0)[0]
    # per-pixel min depth and FIRST index attaining it
    dmin = np.full(P, np.inf, np.float32)
    dmin[nonempty] = np.minimum.reduceat(fb.depth, starts[nonempty])
    pix_of_frag = np.repeat(np.arange(P, dtype=np.int64), n)
    idx = np.arange(fb.depth.shape[0], dtype=np.int64)
    key = np.where(fb.depth == dmin[pix_of_frag], idx, np.int64(1) << 40)
    imin = np.zeros(P, np.int64)
    imin[nonempty] = np.minimum.reduceat(key, starts[nonempty])
    k = (rng.random(chosen.size) * (n[chosen] - 1)).astype(np.int64)
    k = np.minimum(k, n[chosen] - 2)
    j = starts[chosen] + k
    j = np.where(j >= imin[chosen], j + 1, j)
    fb.depth[j] = fb.depth[imin[chosen]]
    return int(chosen.size)
