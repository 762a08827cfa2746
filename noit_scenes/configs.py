"""The five seeded workloads of BASELINE.json (`configs[0..4]` = cfg1..cfg5) and the MLP weights.

INPUT GENERATION ONLY (see raster.py).  The scenes stand in for the paper's ten 3-D test scenes
(§4, Table 2 :157-171), which are not available; what is taken from the paper is
shape only: 1080p frames, maximum depth complexity 12..136, high opacity variation.

All randomness comes from numpy.random.default_rng(seed); the draw order inside each function
is fixed and is part of the recipe (DESIGN.md §"Input recipe").
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .raster import (KIND_ELLIPSE, KIND_QUAD, KIND_RECT, REGION_ALL, REGION_DETAIL,
                     REGION_SMOOTH, FragBuf, Primitives, count_fragments, inject_front_ties,
                     rasterize)

MLP_PARAMS = 5 * 32 + 32 + 32 * 16 + 16 + 16 * 3 + 3   # 771 (5 -> 32 -> 16 -> 3)


def mlp_weights(seed: int) -> np.ndarray:
    """771 fp32 parameters, order W1[32][5], b1[32], W2[16][32], b2[16], W3[3][16], b3[3].

    Seeded random init (no trained weights exist here, BASELINE.json north_star; SURVEY.md
    §8(c) A7): each tensor U(-1/sqrt(fan_in), +1/sqrt(fan_in)) drawn as float64 in the order
    W1, b1, W2, b2, W3, b3 and cast to fp32; b3 += 0.25 so the output ReLU is mostly alive.
    """
    rng = np.random.default_rng(seed)
    parts = []
    for fan_in, fan_out in ((5, 32), (32, 16), (16, 3)):
        bound = 1.0 / np.sqrt(fan_in)
        w = rng.uniform(-bound, bound, size=(fan_out, fan_in))
        b = rng.uniform(-bound, bound, size=(fan_out,))
        parts += [w.ravel(), b]
    parts[-1] = parts[-1] + 0.25
    out = np.concatenate(parts).astype(np.float32)
    assert out.shape[0] == MLP_PARAMS
    return out


# cfg3/cfg4 centre mixture: 70 % of the ellipses around 4 Gaussian hot-spots of unequal weight,
# 30 % uniform.  Chosen (by looking at count histograms only) so that the per-pixel count has a
# heavy tail that reaches the 128 cap: median ~14, p90 ~61, p99 ~112, max 128 at mean 24.
HOTSPOT_SHARE = 0.7
HOTSPOT_WEIGHTS = (0.45, 0.30, 0.15, 0.10)
HOTSPOT_SIGMA = 0.04


@dataclass
class Scene:
    """One frame's inputs: the full-res buffer plus (cfg4) the coarse buffers."""
    name: str
    full: FragBuf
    half: FragBuf | None = None
    quarter: FragBuf | None = None
    weights: np.ndarray | None = None       # 771 fp32
    mlp_precision: int = 0                  # 0 = fp32 weights, 1 = bf16-rounded weights
    background: tuple = (0.2, 0.3, 0.4)
    meta: dict = field(default_factory=dict)


# ----------------------------------------------------------------------------------------------
# primitive generators
# ----------------------------------------------------------------------------------------------
def _screen_prims(rng: np.random.Generator, n: int, W: int, H: int, kinds: str, centres: str,
                  alpha_dist: str, half_extent=(8.0, 40.0)) -> Primitives:
    """n rectangles / rotated ellipses with planar depth and a linear colour gradient.

    Draw order (all vectorised draws of length n, in this order): kind, centre mixture choice,
    centre x, centre y, hot-spot id, hot-spot jitter x, y, half extents (2), angle, z0, gx, gy,
    base colour (3), colour gradients (3x2), alpha.
    """
    P = Primitives.empty(n)
    u_kind = rng.random(n)
    if kinds == "rect":
        P.kind[:] = KIND_RECT
    elif kinds == "ellipse":
        P.kind[:] = KIND_ELLIPSE
    else:
        P.kind[:] = np.where(u_kind < 0.5, KIND_RECT, KIND_ELLIPSE)
    u_mix = rng.random(n)
    cx = rng.uniform(0.0, W, n)
    cy = rng.uniform(0.0, H, n)
    hot = rng.choice(4, n, p=HOTSPOT_WEIGHTS)
    jx = rng.normal(0.0, HOTSPOT_SIGMA * W, n)
    jy = rng.normal(0.0, HOTSPOT_SIGMA * W, n)
    if centres == "hotspots":
        # 4 hot-spot centres are themselves the first 8 uniforms of a child stream
        hs = np.random.default_rng(rng.integers(0, 2 ** 31)).uniform(0.15, 0.85, (4, 2))
        use = u_mix < HOTSPOT_SHARE
        cx = np.where(use, hs[hot, 0] * W + jx, cx)
        cy = np.where(use, hs[hot, 1] * H + jy, cy)
    hx = rng.uniform(half_extent[0], half_extent[1], n)
    hy = rng.uniform(half_extent[0], half_extent[1], n)
    th = rng.uniform(0.0, np.pi, n)
    z0 = rng.uniform(0.1, 0.9, n)
    gx = rng.uniform(-0.2, 0.2, n)
    gy = rng.uniform(-0.2, 0.2, n)
    base = rng.uniform(0.0, 1.0, (n, 3))
    cgrad = rng.uniform(-0.2, 0.2, (n, 3, 2))
    if alpha_dist == "uniform":
        alpha = rng.uniform(0.1, 0.9, n)
    else:
        alpha = np.clip(rng.beta(0.5, 0.5, n), 0.02, 0.98)
    P.geom[:, 0], P.geom[:, 1], P.geom[:, 2], P.geom[:, 3] = cx, cy, hx, hy
    P.geom[:, 4], P.geom[:, 5] = np.cos(th), np.sin(th)
    # z = z0 + gx*(px-cx)/W + gy*(py-cy)/H
    P.zplane[:, 0] = z0 - gx * cx / W - gy * cy / H
    P.zplane[:, 1] = gx / W
    P.zplane[:, 2] = gy / H
    for k in range(3):
        P.cplane[:, k, 0] = base[:, k] - cgrad[:, k, 0] * cx / W - cgrad[:, k, 1] * cy / H
        P.cplane[:, k, 1] = cgrad[:, k, 0] / W
        P.cplane[:, k, 2] = cgrad[:, k, 1] / H
    P.alpha[:] = alpha
    P.region[:] = REGION_ALL
    P.update_bbox()
    return P


def _calibrate(prims: Primitives, W: int, H: int, cap: int, lo_hi, smooth_tiles=None,
               r_cal: int = 4) -> Primitives:
    """One global size factor, by bisection, so that mean fragments/pixel lands in lo_hi."""
    lo, hi = lo_hi
    target = 0.5 * (lo + hi)

    def mean_at(s, r):
        c = count_fragments(prims.scaled(s), W, H, r=r, cap=cap, smooth_tiles=smooth_tiles)
        return float(c.mean())

    a, b = 0.05, 1.0
    while mean_at(b, r_cal) < target and b < 256:
        b *= 2.0
    for _ in range(14):
        m = 0.5 * (a + b)
        if mean_at(m, r_cal) < target:
            a = m
        else:
            b = m
    s = 0.5 * (a + b)
    if r_cal != 1:
        # confirm at full resolution; nudge with a few secant-like steps if outside the band
        for _ in range(4):
            got = mean_at(s, 1)
            if lo <= got <= hi:
                break
            s *= np.sqrt(target / max(got, 1e-9))
    return prims.scaled(s)


# ----------------------------------------------------------------------------------------------
# cfg1..cfg4
# ----------------------------------------------------------------------------------------------
def cfg1(seed: int = 0) -> Scene:
    """64x64, 16 rectangles, <=16 frags/px, RGBA fp32, MLP fp32 (BASELINE.json configs[0])."""
    W = H = 64
    rng = np.random.default_rng(seed)
    prims = _screen_prims(rng, 16, W, H, "rect", "uniform", "uniform")
    fb = rasterize(prims, W, H, 1, cap=16, color_dtype=np.float32)
    return Scene("cfg1", fb, weights=mlp_weights(seed), mlp_precision=0,
                 meta=dict(seed=seed, prims=16))


def cfg2(seed: int = 0, W: int = 1280, H: int = 720, n_prims: int = 128) -> Scene:
    """720p, 128 quads/ellipses, mean ~8, max 32, RGBA fp16, bf16 weights (configs[1])."""
    rng = np.random.default_rng(seed)
    prims = _screen_prims(rng, n_prims, W, H, "mixed", "uniform", "uniform")
    prims = _calibrate(prims, W, H, 32, (7.6, 8.4))
    fb = rasterize(prims, W, H, 1, cap=32, color_dtype=np.float16)
    return Scene("cfg2", fb, weights=mlp_weights(seed), mlp_precision=1,
                 meta=dict(seed=seed, prims=n_prims))


def _cfg3_prims(rng, W, H, n_prims):
    return _screen_prims(rng, n_prims, W, H, "ellipse", "hotspots", "beta")


def cfg3(seed: int = 0, W: int = 1920, H: int = 1080, n_prims: int = 512,
         mean_band=(23.0, 25.0), cap: int = 128, coarse: bool = False) -> Scene:
    """1080p, 512 ellipses, mean ~24, max 128, Beta(.5,.5) alpha, 10% front ties (configs[2]).

    With coarse=True the half- and quarter-resolution buffers are rasterised from the same
    calibrated primitive list as well (used by the whole-path benchmark step).
    """
    rng = np.random.default_rng(seed)
    prims = _cfg3_prims(rng, W, H, n_prims)
    prims = _calibrate(prims, W, H, cap, mean_band)
    fb = rasterize(prims, W, H, 1, cap=cap, color_dtype=np.float16)
    nt = inject_front_ties(fb, rng, 0.10)
    sc = Scene("cfg3", fb, weights=mlp_weights(seed), mlp_precision=1,
               meta=dict(seed=seed, prims=n_prims, tie_pixels=nt))
    if coarse:
        sc.half = rasterize(prims, W, H, 2, cap=cap, color_dtype=np.float16)
        sc.quarter = rasterize(prims, W, H, 4, cap=cap, color_dtype=np.float16)
    return sc


def smooth_tile_mask(rng: np.random.Generator, Tx: int, Ty: int, lo=0.47, hi=0.53) -> np.ndarray:
    """Seeded union of tile-aligned blocks covering 50 +- 3 % of the 64-px tiles."""
    m = np.zeros((Ty, Tx), bool)
    for _ in range(10000):
        f = m.mean()
        if lo <= f <= hi:
            break
        bw = int(rng.integers(1, max(2, Tx // 4)))
        bh = int(rng.integers(1, max(2, Ty // 3)))
        x0 = int(rng.integers(0, Tx - bw + 1))
        y0 = int(rng.integers(0, Ty - bh + 1))
        if f < lo:
            trial = m.copy()
            trial[y0:y0 + bh, x0:x0 + bw] = True
            if trial.mean() <= hi:
                m = trial
        else:
            m[y0:y0 + 1, x0:x0 + 1] = False
    return m


def cfg4(seed: int = 0, W: int = 1920, H: int = 1080, n_prims: int = 512,
         mean_band=(23.0, 25.0), cap: int = 128) -> Scene:
    """cfg3 + smooth low-variance regions over ~50 % of the screen, with coarse buffers.

    Tiles flagged smooth are cleared of ellipses and covered by 3 screen-filling quads whose
    colour gradient is <= 0.004 per 64 px (variance below the cfg4 threshold but non-zero).
    The detail regions keep the cfg3 statistics (mean ~24 there).  The half- and quarter-res
    buffers are rasterised from the same primitive list.
    """
    rng = np.random.default_rng(seed)
    Tx, Ty = -(-W // 64), -(-H // 64)
    prims = _cfg3_prims(rng, W, H, n_prims)
    prims.region[:] = REGION_DETAIL
    smooth = smooth_tile_mask(rng, Tx, Ty)
    # calibrate the detail regions alone to the cfg3 band (mean over detail pixels)
    frac_detail = 1.0 - _pixel_fraction(smooth, W, H)
    band = (mean_band[0] * frac_detail, mean_band[1] * frac_detail)
    prims = _calibrate(prims, W, H, cap, band, smooth_tiles=smooth)
    # 3 full-screen smooth quads
    bg = Primitives.empty(3)
    bg.kind[:] = KIND_RECT
    bg.geom[:, 0], bg.geom[:, 1], bg.geom[:, 2], bg.geom[:, 3] = W / 2, H / 2, W, H
    z0 = np.sort(rng.uniform(0.2, 0.8, 3))
    base = rng.uniform(0.25, 0.75, (3, 3))
    cg = rng.uniform(-0.004 / 64.0, 0.004 / 64.0, (3, 3, 2))
    for i in range(3):
        bg.zplane[i] = (z0[i], 0.01 / W, 0.01 / H)
        for k in range(3):
            bg.cplane[i, k] = (base[i, k], cg[i, k, 0], cg[i, k, 1])
    bg.alpha[:] = rng.uniform(0.2, 0.5, 3)
    bg.region[:] = REGION_SMOOTH
    bg.update_bbox()
    allp = _concat(prims, bg)
    full = rasterize(allp, W, H, 1, cap=cap, color_dtype=np.float16, smooth_tiles=smooth)
    # ties only in the detail tiles: a front tie reorders a pixel's layers, which inside a smooth
    # region would be salt-and-pepper noise and no 64-px leaf would survive (DESIGN.md recipe)
    ys = np.minimum(np.arange(H) // 64, Ty - 1)
    xs = np.minimum(np.arange(W) // 64, Tx - 1)
    detail_px = ~smooth[ys[:, None], xs[None, :]].reshape(-1)
    nt = inject_front_ties(full, rng, 0.10, pixel_mask=detail_px)
    half = rasterize(allp, W, H, 2, cap=cap, color_dtype=np.float16, smooth_tiles=smooth)
    quarter = rasterize(allp, W, H, 4, cap=cap, color_dtype=np.float16, smooth_tiles=smooth)
    return Scene("cfg4", full, half, quarter, weights=mlp_weights(seed), mlp_precision=1,
                 meta=dict(seed=seed, prims=n_prims, tie_pixels=nt,
                           smooth_tile_fraction=float(smooth.mean()), smooth_tiles=smooth))


def _pixel_fraction(tiles: np.ndarray, W: int, H: int) -> float:
    ys = np.minimum(np.arange(H) // 64, tiles.shape[0] - 1)
    xs = np.minimum(np.arange(W) // 64, tiles.shape[1] - 1)
    return float(tiles[ys[:, None], xs[None, :]].mean())


def _concat(a: Primitives, b: Primitives) -> Primitives:
    return Primitives(*[np.concatenate([getattr(a, f), getattr(b, f)]) for f in
                        ("kind", "geom", "edges", "bbox", "zplane", "cplane", "alpha", "region")])


# ----------------------------------------------------------------------------------------------
# cfg5: world-space quads under a moving perspective camera
# ----------------------------------------------------------------------------------------------
def perspective(fovy_deg: float, aspect: float, near: float, far: float) -> np.ndarray:
    """Projection with clip z/w in (0,1) (near -> 0, far -> 1), camera looking down +z,
    x right, y DOWN on screen (no y flip)."""
    f = 1.0 / np.tan(np.radians(fovy_deg) / 2.0)
    Pm = np.zeros((4, 4))
    Pm[0, 0] = f / aspect
    Pm[1, 1] = f
    Pm[2, 2] = far / (far - near)
    Pm[2, 3] = -far * near / (far - near)
    Pm[3, 2] = 1.0
    return Pm


def view_matrix(pos: np.ndarray, yaw: float, pitch: float) -> np.ndarray:
    cy, sy = np.cos(yaw), np.sin(yaw)
    cp, sp = np.cos(pitch), np.sin(pitch)
    Ry = np.array([[cy, 0, -sy], [0, 1, 0], [sy, 0, cy]])
    Rx = np.array([[1, 0, 0], [0, cp, sp], [0, -sp, cp]])
    R = Rx @ Ry
    V = np.eye(4)
    V[:3, :3] = R
    V[:3, 3] = -R @ pos
    return V


@dataclass
class Sequence:
    """cfg5: per-frame view-projection matrices and the world-space quads."""
    width: int
    height: int
    vp: list                # float64 [4,4] per frame
    corners: np.ndarray     # [n, 4, 3] world-space quad corners (convex, planar)
    colors: np.ndarray      # [n, 4, 3] per-corner colours (corner 3 follows from planarity)
    alpha: np.ndarray       # [n]
    weights: np.ndarray
    cap: int
    mlp_precision: int = 1
    background: tuple = (0.2, 0.3, 0.4)
    depth_threshold: float = 1e-3

    def reproject_matrix(self, t: int) -> np.ndarray:
        """M = VP_{t-1} . VP_t^{-1} in float64, cast to fp32, row-major."""
        return (self.vp[t - 1] @ np.linalg.inv(self.vp[t])).astype(np.float32)

    def frame_prims(self, t: int) -> Primitives:
        return _project_quads(self.corners, self.colors, self.alpha, self.vp[t],
                              self.width, self.height)

    def frame(self, t: int) -> FragBuf:
        return rasterize(self.frame_prims(t), self.width, self.height, 1, cap=self.cap,
                         color_dtype=np.float16)


def _project_quads(corners, colors, alpha, VP, W, H) -> Primitives:
    n = corners.shape[0]
    P = Primitives.empty(n)
    P.kind[:] = KIND_QUAD
    hom = np.concatenate([corners, np.ones((n, 4, 1))], axis=2) @ VP.T      # [n,4,4]
    w = hom[..., 3]
    ok = (w > 1e-6).all(axis=1)
    ndc = hom[..., :3] / np.where(w[..., None] > 1e-6, w[..., None], 1.0)
    sx = (ndc[..., 0] + 1.0) * 0.5 * W
    sy = (ndc[..., 1] + 1.0) * 0.5 * H
    for i in range(n):
        if not ok[i]:
            P.bbox[i] = (0, 0, -1, -1)          # behind the camera: draws nothing
            continue
        xs, ys = sx[i], sy[i]
        area = 0.0
        for k in range(4):
            k2 = (k + 1) % 4
            area += xs[k] * ys[k2] - xs[k2] * ys[k]
        sgn = 1.0 if area >= 0 else -1.0
        for k in range(4):
            k2 = (k + 1) % 4
            ex, ey = xs[k2] - xs[k], ys[k2] - ys[k]
            # inside (left of every edge for positive area): ex*(py-ys) - ey*(px-xs) >= 0
            P.edges[i, k] = (-ey * sgn, ex * sgn, (ey * xs[k] - ex * ys[k]) * sgn)
        P.bbox[i] = (xs.min(), ys.min(), xs.max(), ys.max())
        # affine planes through projected vertices 0,1,3 (z_ndc is affine in screen space
        # for a planar primitive; colour uses the same affine fit)
        A = np.array([[1, xs[0], ys[0]], [1, xs[1], ys[1]], [1, xs[3], ys[3]]])
        if abs(np.linalg.det(A)) < 1e-9:
            P.bbox[i] = (0, 0, -1, -1)
            continue
        P.zplane[i] = np.linalg.solve(A, ndc[i, [0, 1, 3], 2])
        for k in range(3):
            P.cplane[i, k] = np.linalg.solve(A, colors[i, [0, 1, 3], k])
    P.alpha[:] = alpha
    P.region[:] = REGION_ALL
    return P


def cfg5(seed: int = 0, W: int = 3840, H: int = 2160, n_quads: int = 256, n_frames: int = 8,
         mean_band=(11.0, 13.0), cap: int = 64, max_motion: float = 0.02) -> Sequence:
    """4K, 8 frames, 256 world-space quads, mean ~12, camera path <= 2 % screen motion/frame.

    Draw order: quad centres (3n), edge directions (2 x 3n), half sizes (2n), colours (4x3 n),
    alpha (n), camera translation steps (3 per frame), yaw/pitch steps (2 per frame).
    """
    rng = np.random.default_rng(seed)
    near, far = 0.1, 100.0
    proj = perspective(60.0, W / H, near, far)
    ctr = np.stack([rng.uniform(-6, 6, n_quads), rng.uniform(-3.5, 3.5, n_quads),
                    rng.uniform(4.0, 14.0, n_quads)], axis=1)
    e1 = rng.normal(size=(n_quads, 3))
    e2 = rng.normal(size=(n_quads, 3))
    e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
    e2 -= (e2 * e1).sum(1, keepdims=True) * e1
    e2 /= np.linalg.norm(e2, axis=1, keepdims=True)
    hs = rng.uniform(0.5, 1.5, (n_quads, 2))
    cols = rng.uniform(0.0, 1.0, (n_quads, 4, 3))
    alpha = rng.uniform(0.1, 0.9, n_quads)
    dpos = rng.normal(size=(n_frames, 3))
    dang = rng.normal(size=(n_frames, 2))

    def corners_at(s):
        a = e1 * (hs[:, :1] * s)
        b = e2 * (hs[:, 1:] * s)
        return np.stack([ctr - a - b, ctr + a - b, ctr + a + b, ctr - a + b], axis=1)

    vp0 = proj @ view_matrix(np.zeros(3), 0.0, 0.0)

    def mean_at(s, r):
        pr = _project_quads(corners_at(s), cols, alpha, vp0, W, H)
        return float(count_fragments(pr, W, H, r=r, cap=cap).mean())

    target = 0.5 * (mean_band[0] + mean_band[1])
    a_, b_ = 0.05, 1.0
    while mean_at(b_, 8) < target and b_ < 64:
        b_ *= 2
    for _ in range(14):
        m = 0.5 * (a_ + b_)
        if mean_at(m, 8) < target:
            a_ = m
        else:
            b_ = m
    s = 0.5 * (a_ + b_)
    corners = corners_at(s)

    # camera path: random step directions, scaled so that the largest projected corner
    # displacement between consecutive frames is <= max_motion * W
    vps = [vp0]
    pos, yaw, pitch = np.zeros(3), 0.0, 0.0
    hom = np.concatenate([corners.reshape(-1, 3), np.ones((n_quads * 4, 1))], axis=1)

    def screen(vp):
        h = hom @ vp.T
        wv = np.maximum(h[:, 3], 1e-6)
        return np.stack([(h[:, 0] / wv + 1) * 0.5 * W, (h[:, 1] / wv + 1) * 0.5 * H], 1)

    for t in range(1, n_frames):
        step = 1.0
        for _ in range(40):
            p2 = pos + dpos[t] * 0.05 * step
            y2 = yaw + dang[t, 0] * 0.01 * step
            q2 = pitch + dang[t, 1] * 0.01 * step
            vp = proj @ view_matrix(p2, y2, q2)
            a0, a1 = screen(vps[-1]), screen(vp)
            vis = ((a0[:, 0] > -W) & (a0[:, 0] < 2 * W) & (a0[:, 1] > -H) & (a0[:, 1] < 2 * H))
            disp = np.abs(a1 - a0)[vis].max() if vis.any() else 0.0
            if disp <= max_motion * W:
                break
            step *= 0.7
        pos, yaw, pitch = p2, y2, q2
        vps.append(vp)
    return Sequence(W, H, vps, corners, cols, alpha, mlp_weights(seed), cap)
