"""GPU parity for the adjacent steps (`-m gpu`): S6 quadtree, S7 adaptive resolve, S8
reprojection, S9 fallback resolve, and the ABI's error behaviour."""
import numpy as np
import pytest
import torch

import noit_scenes
from noit_scenes.raster import FragBuf
import oracle
from test_parity_gpu import (BG, EPS32, K_MLP, check_resolve, close, mlp_magnitude, noit,  # noqa: F401
                             random_fb, u32)

pytestmark = pytest.mark.gpu


def qt_equal(got, ref):
    assert np.array_equal(u32(got["tile_mask"]), ref["tile_mask"])
    assert np.array_equal(got["cell_level"].cpu().numpy(), ref["cell_level"])
    assert np.array_equal(u32(got["hist"]), ref["hist"])


# -------------------------------------------------------------------------------------------
# S6
# -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("W,H", [(64, 64), (200, 136), (1920, 1080), (65, 7)])
@pytest.mark.parametrize("metric", [0, 1])
def test_quadtree_random_images(noit, W, H, metric):
    rng = np.random.default_rng(W * 7 + H + metric)
    # very smooth field + 16-px blocks of noise of three amplitudes, so that every level occurs
    yy, xx = np.mgrid[0:H, 0:W]
    img = np.zeros((H, W, 4), np.float32)
    for c in range(3):
        img[..., c] = 0.5 + 0.004 * np.sin(xx / (300.0 + 50 * c)) * np.cos(yy / 400.0)
    noise = rng.random((H, W, 3)).astype(np.float32)
    sel = (rng.random((-(-H // 16), -(-W // 16))) < 0.12).repeat(16, 0).repeat(16, 1)[:H, :W]
    amp = rng.choice([0.01, 0.05, 0.6], size=(-(-H // 16), -(-W // 16))).astype(np.float32)
    amp = amp.repeat(16, 0).repeat(16, 1)[:H, :W]
    img[..., :3] += (sel * amp)[..., None] * (noise - 0.5)
    img[..., 3] = rng.random((H, W))
    img = np.ascontiguousarray(img.reshape(-1, 4))
    ctx = noit.Noit()
    for thr, cthr in ((6, 0.02), (0, 0.0), (400, 0.2)):
        got = ctx.quadtree(torch.from_numpy(img).cuda(), W, H, metric, thr, cthr)
        ref = oracle.quadtree(img, W, H, metric, thr, cthr)
        qt_equal(got, ref)
    levels = set(np.unique(oracle.quadtree(img, W, H, metric, 6, 0.02)["cell_level"]).tolist())
    if W >= 1920 and metric == 0:
        assert levels == {0, 1, 2, 3}


@pytest.mark.parametrize("W,H", [(200, 136), (1920, 1080), (65, 7)])
@pytest.mark.parametrize("metric", [0, 1])
def test_quadtree_out_of_range_pixels(noit, W, H, metric):
    """The resolve's ReLU output is unbounded above (A11) and is what S6 consumes: colours below 0
    and above 1 (the +-2.0 spikes of the first version of test_quadtree_random_images, plus whole
    blocks outside [0, 1]) must give the oracle's masks bit for bit -- both sides quantise
    q = rint(255 * clamp(c, 0, 1)) for the variance metric and use the raw colour in the corner metric.
    The oracle's clamp is pinned on the CPU (test_quadtree_quantiser_clamps_out_of_range_colours)."""
    rng = np.random.default_rng(W * 11 + H + metric)
    yy, xx = np.mgrid[0:H, 0:W]
    img = np.zeros((H, W, 4), np.float32)
    for c in range(3):
        img[..., c] = 0.5 + 0.3 * np.sin(xx / (40.0 + 10 * c)) * np.cos(yy / 55.0)
    img[..., :3] += (rng.random((H, W, 3)) < 0.002) * 2.0 - (rng.random((H, W, 3)) < 0.002) * 2.0
    blocks = rng.choice([0.0, 0.0, 0.0, 1.5, -0.7], size=(-(-H // 32), -(-W // 32))).astype(np.float32)
    img[..., :3] += blocks.repeat(32, 0).repeat(32, 1)[:H, :W, None]
    img[..., 3] = rng.random((H, W))
    assert W < 128 or ((img[..., :3] < 0).any() and (img[..., :3] > 1).any())
    img = np.ascontiguousarray(img.reshape(-1, 4))
    ctx = noit.Noit()
    for thr, cthr in ((6, 0.02), (0, 0.0), (400, 0.2)):
        qt_equal(ctx.quadtree(torch.from_numpy(img).cuda(), W, H, metric, thr, cthr),
                 oracle.quadtree(img, W, H, metric, thr, cthr))
    if W >= 128:
        q16 = ctx.quadtree16(torch.from_numpy(img).cuda(), W, H, metric, 6, 0.02)
        qt_equal(q16, oracle.quadtree16(img, W, H, metric, 6, 0.02))


def test_quadtree_constant_image(noit):
    W, H = 300, 200
    img = np.tile(np.asarray([0.3, 0.6, 0.9, 1.0], np.float32), (W * H, 1))
    got = noit.Noit().quadtree(torch.from_numpy(img).cuda(), W, H)
    assert int(got["tile_mask"].abs().sum()) == 0
    assert u32(got["hist"]).tolist() == [5 * 4, 0, 0, 0]


def test_quadtree_on_resolved_cfg1(noit, cfg1_scene):
    sc = cfg1_scene
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    final = ctx.resolve(noit.DeviceFragBuf.from_host(sc.full), BG)["final"]
    for metric in (0, 1):
        got = ctx.quadtree(final, 64, 64, metric, 6, 0.02)
        qt_equal(got, oracle.quadtree(final.cpu().numpy(), 64, 64, metric, 6, 0.02))   # same image (A16)


# -------------------------------------------------------------------------------------------
# S7
# -------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg4_small():
    return noit_scenes.cfg4(0, W=448, H=264, n_prims=96, mean_band=(10.0, 12.0), cap=64)


def run_adaptive(noit, sc, l2l=(2, 1, 0, 0), thr=6):
    fb, hb, qb = (noit.DeviceFragBuf.from_host(b) for b in (sc.full, sc.half, sc.quarter))
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    plain = ctx.resolve(fb, BG)
    qt = ctx.quadtree(plain["final"], fb.width, fb.height, 0, thr)
    got = ctx.resolve(fb, BG, half=hb, quarter=qb, cell_level=qt["cell_level"], level_to_lod=l2l)
    cell = qt["cell_level"].cpu().numpy()
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    ref = oracle.resolve(sc.full, w_eff, BG, half=sc.half, quarter=sc.quarter, cell_level=cell,
                         level_to_lod=l2l)
    return plain, got, ref, cell


def test_adaptive_resolve_small(noit, cfg4_small):
    sc = cfg4_small
    plain, got, ref, cell = run_adaptive(noit, sc)
    assert {0, 1}.issubset(set(np.unique(cell).tolist())) or 0 in cell      # coarse leaves exist
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
    # features of coarse pixels are interpolated: bound the MLP error with a generous magnitude
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    lay = oracle.build_features(sc.full)
    mag = mlp_magnitude(w_eff, np.maximum(lay["features"], [[64, 1, 1, 1, 1]]))
    extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
    for k in ("trans", "final"):
        close(got[k].cpu().numpy(), ref[k], extra=extra)
        assert np.max(np.abs(got[k].cpu().numpy()[:, :3] - ref[k][:, :3])) <= 2e-3
    # all levels -> lod 0 is the plain resolve (O7 pin).  The plain frame runs in the staged
    # kernel (4 lanes per pixel), the adaptive frame in the one-thread-per-pixel kernel: same
    # selection, different fp32 summation order => layer-1 depth bitwise, colours to tolerance.
    _, got0, _, _ = run_adaptive(noit, sc, l2l=(0, 0, 0, 0))
    assert torch.equal(got0["depth1"], plain["depth1"])
    for k in ("trans", "final"):
        close(got0[k].cpu().numpy(), plain[k].cpu().numpy().astype(np.float64), extra=extra)


def test_adaptive_resolve_ties_in_the_coarse_buffers(noit):
    """Exact front depth ties INSIDE the half and quarter buffers (the generator injects them into
    the full buffer only): the pre-pass's own selection must apply the index tie rule (O1 on the
    coarse lists, A19), for both colour orders of the tied pair."""
    import copy
    from noit_scenes.raster import inject_front_ties
    sc = copy.deepcopy(noit_scenes.cfg4(5, W=448, H=264, n_prims=96, mean_band=(10.0, 12.0), cap=64))
    rng = np.random.default_rng(55)
    assert inject_front_ties(sc.half, rng, 0.5) > 1000 and inject_front_ties(sc.quarter, rng, 0.5) > 300
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    mag = mlp_magnitude(w_eff, np.maximum(oracle.build_features(sc.full)["features"], [[64, 1, 1, 1, 1]]))
    extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
    for l2l, thr in (((2, 1, 0, 0), 6), ((2, 2, 1, 1), 10 ** 9), ((1, 1, 1, 1), 6)):
        _, got, ref, cell = run_adaptive(noit, sc, l2l=l2l, thr=thr)
        assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
        for k in ("trans", "final"):
            close(got[k].cpu().numpy(), ref[k], extra=extra)
    # the frame-global control reads the same coarse buffers through the same pre-pass
    fb, hb, qb = (noit.DeviceFragBuf.from_host(b) for b in (sc.full, sc.half, sc.quarter))
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    forced = torch.tensor([2.0, 0.5, 0.25], dtype=torch.float32, device="cuda")
    g = ctx.resolve(fb, BG, half=hb, quarter=qb, pass_scales=forced)
    r = oracle.resolve_global(sc.full, sc.half, sc.quarter, w_eff, BG, 1, 2)
    for k in ("trans", "final"):
        close(g[k].cpu().numpy(), r[k], extra=extra)


def test_adaptive_resolve_ragged_size(noit):
    """Width not a multiple of 8 (cells cut by the right edge), P not a multiple of 32 (last tile
    partial, tiles wrap rows in the middle of a cell): the per-tile lod summary of the pre-pass
    must agree with the per-pixel levels the oracle uses."""
    sc = noit_scenes.cfg4(3, W=333, H=150, n_prims=64, mean_band=(8.0, 10.0), cap=48)
    assert sc.full.width % 8 and sc.full.num_pixels % 32
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    mag = mlp_magnitude(w_eff, np.maximum(oracle.build_features(sc.full)["features"], [[64, 1, 1, 1, 1]]))
    extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
    for l2l, thr in (((2, 1, 0, 0), 6), ((2, 2, 1, 0), 6), ((1, 1, 1, 1), 6), ((2, 1, 0, 0), 10 ** 9)):
        _, got, ref, cell = run_adaptive(noit, sc, l2l=l2l, thr=thr)
        assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
        for k in ("trans", "final"):
            close(got[k].cpu().numpy(), ref[k], extra=extra)
            assert np.max(np.abs(got[k].cpu().numpy()[:, :3] - ref[k][:, :3])) <= 2e-3


def test_adaptive_all_coarse(noit, cfg4_small):
    """Force every leaf coarse (huge threshold => all 64-leaves => quarter res everywhere)."""
    sc = cfg4_small
    _, got, ref, cell = run_adaptive(noit, sc, thr=10 ** 9)
    assert set(np.unique(cell).tolist()) == {0}
    for k in ("trans", "final"):
        assert np.max(np.abs(got[k].cpu().numpy() - ref[k])) <= 2e-3
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])


# -------------------------------------------------------------------------------------------
# S8 / S9
# -------------------------------------------------------------------------------------------
def rand_prev(rng, W, H):
    P = W * H
    return (rng.random((P, 4)).astype(np.float32), rng.uniform(0.05, 0.95, P).astype(np.float32))


def check_reproject(noit, W, H, M, thr, prev_t, prev_d, cur_d):
    ctx = noit.Noit()
    got = ctx.reproject(W, H, M, thr, BG, torch.from_numpy(prev_t).cuda(), torch.from_numpy(prev_d).cuda(),
                        torch.from_numpy(cur_d).cuda())
    ref = oracle.reproject(W, H, M, thr, BG, prev_t, prev_d, cur_d)
    acc = got["accept"].cpu().numpy()
    assert np.array_equal(acc, ref["accept"])                                  # bit-exact mask
    n = int(got["reject_count"].item())
    assert n == ref["reject_count"]
    assert np.array_equal(np.sort(u32(got["reject_list"])[:n]), np.sort(ref["reject_list"]))
    m = acc.astype(bool)
    assert np.array_equal(got["trans"].cpu().numpy()[m], ref["trans"][m])      # bit copies
    assert np.array_equal(got["depth"].cpu().numpy()[m], ref["depth"][m])
    close(got["final"].cpu().numpy()[m], ref["final"][m])
    assert not got["trans"].cpu().numpy()[~m].any()                            # rejected: untouched
    return got, ref


def test_reproject_identity_and_shift(noit):
    rng = np.random.default_rng(21)
    W, H = 333, 77
    prev_t, prev_d = rand_prev(rng, W, H)
    got, _ = check_reproject(noit, W, H, np.eye(4, dtype=np.float32), 1e-3, prev_t, prev_d, prev_d)
    assert int(got["reject_count"].item()) == 0
    assert np.array_equal(got["trans"].cpu().numpy(), prev_t)
    M = np.eye(4, dtype=np.float32)
    M[0, 3] = 2.0 * 5 / W                                                      # 5-pixel NDC shift
    got, ref = check_reproject(noit, W, H, M, 2.0, prev_t, prev_d, prev_d)
    assert ref["reject_count"] >= 4 * H


def test_reproject_perspective_path(noit):
    rng = np.random.default_rng(22)
    W, H = 640, 360
    proj = noit_scenes.perspective(60.0, W / H, 0.1, 100.0)
    vp0 = proj @ noit_scenes.view_matrix(np.zeros(3), 0.0, 0.0)
    vp1 = proj @ noit_scenes.view_matrix(np.asarray([0.05, -0.02, 0.03]), 0.004, -0.003)
    M = (vp0 @ np.linalg.inv(vp1)).astype(np.float32)
    prev_t, _ = rand_prev(rng, W, H)
    yy, xx = np.mgrid[0:H, 0:W]
    prev_d = (0.97 + 0.02 * np.sin(xx / 50.0) * np.cos(yy / 40.0)).astype(np.float32).reshape(-1)
    prev_d[rng.random(W * H) < 0.05] = 1.0
    got, ref = check_reproject(noit, W, H, M, 1e-3, prev_t, prev_d, prev_d)
    frac = ref["reject_count"] / (W * H)
    assert 0.0 < frac < 1.0
    Mneg = M.copy()
    Mneg[3] = -Mneg[3]                                                         # w <= 0 everywhere
    got, ref = check_reproject(noit, W, H, Mneg, 1e-3, prev_t, prev_d, prev_d)
    assert ref["reject_count"] == W * H


def test_reproject_mode_b_current_depth_differs(noit):
    """Reading A21 mode B: the caller has the CURRENT first-layer depth (a depth-only scan), so
    cur_depth != prev_depth: the transform takes d from cur_depth, the disocclusion test compares
    d_e with prev_depth at the fetched pixel.  Perspective motion, both filters, a third of the
    pixels with a depth change beyond tau."""
    rng = np.random.default_rng(29)
    W, H = 517, 203
    proj = noit_scenes.perspective(60.0, W / H, 0.1, 100.0)
    vp0 = proj @ noit_scenes.view_matrix(np.zeros(3), 0.0, 0.0)
    vp1 = proj @ noit_scenes.view_matrix(np.asarray([0.04, 0.03, -0.02]), -0.005, 0.002)
    M = (vp0 @ np.linalg.inv(vp1)).astype(np.float32)
    prev_t, _ = rand_prev(rng, W, H)
    yy, xx = np.mgrid[0:H, 0:W]
    prev_d = (0.95 + 0.03 * np.sin(xx / 37.0) * np.cos(yy / 29.0)).astype(np.float32).reshape(-1)
    cur_d = prev_d + rng.choice(np.asarray([0.0, 2e-4, -3e-4, 5e-3], np.float32), W * H)
    cur_d = cur_d.astype(np.float32)
    assert not np.array_equal(cur_d, prev_d)
    got, ref = check_reproject(noit, W, H, M, 1e-3, prev_t, prev_d, cur_d)
    assert 0.15 < ref["reject_count"] / (W * H) < 0.9
    check_reproject_bilinear(noit, W, H, M, 1e-3, prev_t, prev_d, cur_d)


def check_reproject_bilinear(noit, W, H, M, thr, prev_t, prev_d, cur_d):
    """NEXT-4 / O8b: same fixed-order fp32 on both sides -> every output bit-exact; accept,
    reject list and depth equal the nearest filter's."""
    ctx = noit.Noit()
    dev = [torch.from_numpy(a).cuda() for a in (prev_t, prev_d, cur_d)]
    got = ctx.reproject(W, H, M, thr, BG, *dev, filter="bilinear")
    near = ctx.reproject(W, H, M, thr, BG, *dev)
    ref = oracle.reproject_bilinear(W, H, M, thr, BG, prev_t, prev_d, cur_d)
    acc = got["accept"].cpu().numpy()
    assert np.array_equal(acc, ref["accept"])
    assert np.array_equal(acc, near["accept"].cpu().numpy())
    n = int(got["reject_count"].item())
    assert n == ref["reject_count"]
    assert np.array_equal(np.sort(u32(got["reject_list"])[:n]), np.sort(ref["reject_list"]))
    m = acc.astype(bool)
    assert np.array_equal(got["trans"].cpu().numpy()[m], ref["trans"][m])      # bit-exact lerps
    assert np.array_equal(got["depth"].cpu().numpy()[m], ref["depth"][m])
    close(got["final"].cpu().numpy()[m], ref["final"][m])
    assert not got["trans"].cpu().numpy()[~m].any()
    # where the footprint was not used the value is the nearest fetch, bit for bit
    keep = m & (ref["filtered"] == 0)
    assert np.array_equal(got["trans"].cpu().numpy()[keep], near["trans"].cpu().numpy()[keep])
    return got, ref


def test_reproject_bilinear_subpixel_shift_and_edges(noit):
    rng = np.random.default_rng(23)
    W, H = 333, 77                                                             # ragged sizes, clamped taps
    prev_t, prev_d = rand_prev(rng, W, H)
    flat = np.full(W * H, 0.5, np.float32)
    for (sx, sy) in ((0.0, 0.0), (0.3, -0.6), (-2.25, 1.75), (5.5, 0.0)):
        M = np.eye(4, dtype=np.float32)
        M[0, 3], M[1, 3] = 2.0 * sx / W, 2.0 * sy / H
        _, ref = check_reproject_bilinear(noit, W, H, M, 1e-3, prev_t, flat, flat)
        assert ref["filtered"].sum() == ref["accept"].sum() > 0               # flat depth: all filtered
        # random depths: most footprints straddle a "discontinuity" and keep the nearest pixel
        _, ref = check_reproject_bilinear(noit, W, H, M, 0.2, prev_t, prev_d, prev_d)
        if (sx, sy) != (0.0, 0.0):
            f = ref["filtered"][ref["accept"].astype(bool)]
            assert 0 < f.sum() < f.size
    with pytest.raises(Exception):
        noit.Noit().reproject(W, H, np.eye(4, dtype=np.float32), 1e-3, BG, torch.from_numpy(prev_t).cuda(),
                              torch.from_numpy(flat).cuda(), torch.from_numpy(flat).cuda(), filter=7)


def test_reproject_bilinear_perspective_path(noit):
    rng = np.random.default_rng(24)
    W, H = 640, 360
    proj = noit_scenes.perspective(60.0, W / H, 0.1, 100.0)
    vp0 = proj @ noit_scenes.view_matrix(np.zeros(3), 0.0, 0.0)
    vp1 = proj @ noit_scenes.view_matrix(np.asarray([0.05, -0.02, 0.03]), 0.004, -0.003)
    M = (vp0 @ np.linalg.inv(vp1)).astype(np.float32)
    prev_t, _ = rand_prev(rng, W, H)
    yy, xx = np.mgrid[0:H, 0:W]
    prev_d = (0.97 + 0.02 * np.sin(xx / 50.0) * np.cos(yy / 40.0)).astype(np.float32).reshape(-1)
    prev_d[rng.random(W * H) < 0.05] = 1.0
    _, ref = check_reproject_bilinear(noit, W, H, M, 1e-3, prev_t, prev_d, prev_d)
    acc = ref["accept"].astype(bool)
    assert 0 < ref["filtered"][acc].sum() < acc.sum()


def test_fallback_resolve_on_reject_list(noit):
    """S8 + S9: union of accepted and re-resolved pixels covers the frame exactly once; with a
    negative threshold everything is rejected and the frame equals the plain resolve (layer-1
    depth bitwise; colours to the fp32 tolerance, because the plain frame runs in the staged
    kernel and the listed pixels in the one-thread-per-pixel kernel: same selection, different
    fp32 summation order)."""
    rng = np.random.default_rng(23)
    W, H = 160, 96
    fbh = random_fb(rng, W, H, 24, np.float16)
    w = noit_scenes.mlp_weights(3)
    ctx = noit.Noit(w, 1)
    fb = noit.DeviceFragBuf.from_host(fbh)
    plain = ctx.resolve(fb, BG)
    M = np.eye(4, dtype=np.float32)
    M[0, 3] = 2.0 * 3 / W
    for thr in (0.05, -1.0):
        rp = ctx.reproject(W, H, M, thr, BG, plain["trans"], plain["depth1"], plain["depth1"])
        out = dict(trans=rp["trans"], final=rp["final"], depth1=rp["depth"])
        ctx.resolve(fb, BG, out=out, pixel_list=rp["reject_list"], pixel_count=rp["reject_count"])
        acc = rp["accept"].cpu().numpy().astype(bool)
        n = int(rp["reject_count"].item())
        assert n == int((~acc).sum())
        w_eff = oracle.effective_weights(w, 1)
        ref_rp = oracle.reproject(W, H, M, thr, BG, plain["trans"].cpu().numpy(),
                                  plain["depth1"].cpu().numpy(), plain["depth1"].cpu().numpy())
        ref = dict(trans=ref_rp["trans"], final=ref_rp["final"], depth1=ref_rp["depth"])
        oracle.resolve(fbh, w_eff, BG, pixel_list=ref_rp["reject_list"], out=ref)
        for k in ("trans", "final"):
            assert np.max(np.abs(out[k].cpu().numpy() - ref[k])) <= 2e-3
        rej = ~torch.from_numpy(acc).cuda()                                    # rejected == plain
        lay = oracle.build_features(fbh)
        mag = mlp_magnitude(w_eff, np.maximum(lay["features"], [[64, 1, 1, 1, 1]]))
        extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)[~acc]
        assert torch.equal(out["depth1"][rej], plain["depth1"][rej])
        for k in ("trans", "final"):
            close(out[k][rej].cpu().numpy(), plain[k][rej].cpu().numpy(), extra=extra)
        if thr < 0:
            assert n == W * H


# -------------------------------------------------------------------------------------------
# ABI error behaviour: host-checkable errors come back before any launch
# -------------------------------------------------------------------------------------------
# -------------------------------------------------------------------------------------------
# BASELINE.json configs[3] and configs[4] at FULL size, in the call sequence bench.py times
# -------------------------------------------------------------------------------------------
def test_cfg4_full_size_adaptive_frame(noit):
    """1920x1080 adaptive tiling (cfg4): resolve -> quadtree -> balance -> adaptive resolve."""
    sc = noit_scenes.cfg4(0)
    fb, hb, qb = (noit.DeviceFragBuf.from_host(b) for b in (sc.full, sc.half, sc.quarter))
    W, H = fb.width, fb.height
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    plain = ctx.resolve(fb, BG)
    check_resolve(noit, sc.full, sc.weights, sc.mlp_precision, plain)
    img = plain["final"].cpu().numpy()
    qt = ctx.quadtree(plain["final"], W, H, 0, 6)
    ref_qt = oracle.quadtree(img, W, H, 0, 6)                                  # same image (A16)
    qt_equal(qt, ref_qt)
    coarse = np.isin(ref_qt["cell_level"], (0, 1)).mean()
    assert 0.3 < coarse < 0.6, coarse                                          # ~50 % smooth regions
    bal = ctx.quadtree_balance(qt["tile_mask"], W, H)
    ref_bal = oracle.quadtree_balance(ref_qt["tile_mask"], W, H)
    assert np.array_equal(u32(bal["tile_mask"]), ref_bal["tile_mask"])
    assert np.array_equal(bal["cell_level"].cpu().numpy(), ref_bal["cell_level"])
    assert np.array_equal(u32(bal["hist"]), ref_bal["hist"])
    got = ctx.resolve(fb, BG, half=hb, quarter=qb, cell_level=bal["cell_level"])
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    ref = oracle.resolve(sc.full, w_eff, BG, half=sc.half, quarter=sc.quarter,
                         cell_level=ref_bal["cell_level"])
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
    lay = oracle.build_features(sc.full)
    mag = mlp_magnitude(w_eff, np.maximum(lay["features"], [[64, 1, 1, 1, 1]]))
    extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
    for k in ("trans", "final"):
        close(got[k].cpu().numpy(), ref[k], extra=extra)
        assert np.max(np.abs(got[k].cpu().numpy()[:, :3] - ref[k][:, :3])) <= 2e-3


def run_sequence(noit, seq, n_frames):
    """cfg5's schedule: even frames are resolved, odd frames reuse the previous transparency
    result by reprojection (mode A: cur_depth = prev_depth) and resolve the rejected pixels."""
    W, H = seq.width, seq.height
    ctx = noit.Noit(seq.weights, seq.mlp_precision)
    w_eff = oracle.effective_weights(seq.weights, seq.mlp_precision)
    prev = None
    fractions = []
    for t in range(n_frames):
        fbh = seq.frame(t)
        fb = noit.DeviceFragBuf.from_host(fbh)
        if t % 2 == 0:
            got = ctx.resolve(fb, seq.background)
            check_resolve(noit, fbh, seq.weights, seq.mlp_precision, got,
                          ref=oracle.resolve(fbh, w_eff, seq.background))
            prev = got
            continue
        M = seq.reproject_matrix(t)
        p_t, p_d = prev["trans"].cpu().numpy(), prev["depth1"].cpu().numpy()
        rp = ctx.reproject(W, H, M, seq.depth_threshold, seq.background, prev["trans"], prev["depth1"],
                           prev["depth1"])
        ref_rp = oracle.reproject(W, H, M, seq.depth_threshold, seq.background, p_t, p_d, p_d)
        acc = rp["accept"].cpu().numpy()
        assert np.array_equal(acc, ref_rp["accept"])                           # bit-exact mask
        n = int(rp["reject_count"].item())
        assert n == ref_rp["reject_count"] == int((acc == 0).sum())
        assert np.array_equal(np.sort(u32(rp["reject_list"])[:n]), np.sort(ref_rp["reject_list"]))
        out = dict(trans=rp["trans"], final=rp["final"], depth1=rp["depth"])
        ctx.resolve(fb, seq.background, out=out, pixel_list=rp["reject_list"],
                    pixel_count=rp["reject_count"])
        ref = dict(trans=ref_rp["trans"], final=ref_rp["final"], depth1=ref_rp["depth"])
        oracle.resolve(fbh, w_eff, seq.background, pixel_list=ref_rp["reject_list"], out=ref)
        m = acc.astype(bool)
        assert np.array_equal(out["trans"].cpu().numpy()[m], ref["trans"][m])  # accepted: bit copies
        assert np.array_equal(out["depth1"].cpu().numpy(), ref["depth1"])
        lay = oracle.build_features(fbh)
        mag = mlp_magnitude(w_eff, np.maximum(lay["features"], [[64, 1, 1, 1, 1]]))
        extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
        for k in ("trans", "final"):
            close(out[k].cpu().numpy(), ref[k], extra=extra)
        fractions.append(n / (W * H))
    return fractions


def test_cfg5_sequence_reduced_all_eight_frames(noit):
    """The whole 8-frame schedule of cfg5 on a 960x540 version of the same scene and camera path."""
    seq = noit_scenes.cfg5(0, W=960, H=540)
    fr = run_sequence(noit, seq, 8)
    assert len(fr) == 4 and all(0.0 < f < 0.5 for f in fr), fr


def test_cfg5_full_size_all_eight_frames(noit):
    """BASELINE.json configs[4] as stated: 3840x2160, 8 frames, frames 0/2/4/6 resolved and compared
    element by element, frames 1/3/5/7 reprojected (accept mask, reject set, copies bit-exact) with
    the rejected pixels resolved by S9.  Frames are rasterised one at a time (~25 s each on the host)."""
    seq = noit_scenes.cfg5(0)
    assert (seq.width, seq.height) == (3840, 2160)
    fr = run_sequence(noit, seq, 8)
    assert len(fr) == 4 and all(0.0 < f < 0.5 for f in fr), fr


# -------------------------------------------------------------------------------------------
# NEXT-1: quadtree consistency + demand index (O10)
# -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,W,H,k", [(0, 1920, 1080, 2), (1, 3840, 2160, 2), (2, 40, 40, 2),
                                        (3, 300, 50, 2), (4, 1000, 700, 1), (5, 1000, 700, 5),
                                        (6, 640, 640, 0)])
def test_quadtree_balance_random_masks(noit, seed, W, H, k):
    from test_oracle_pins import _random_valid_masks
    rng = np.random.default_rng(seed)
    Tx, Ty = (W + 63) // 64, (H + 63) // 64
    m = _random_valid_masks(rng, Tx * Ty)
    ref = oracle.quadtree_balance(m, W, H, iterations=k)
    ctx = noit.Noit()
    d_mask = torch.from_numpy(m.view(np.int32).copy()).cuda()
    got = ctx.quadtree_balance(d_mask, W, H, iterations=k)
    got2 = None
    if k == 2:                                         # balanced input: a second call is a no-op
        got2 = ctx.quadtree_balance(d_mask.clone(), W, H, iterations=k)
    assert np.array_equal(u32(got["tile_mask"]), ref["tile_mask"])
    assert np.array_equal(got["tile_level"].cpu().numpy(), ref["tile_level"])
    assert np.array_equal(got["cell_level"].cpu().numpy(), ref["cell_level"])
    assert np.array_equal(u32(got["hist"]), ref["hist"])
    assert np.max(np.abs(got["scales"].cpu().numpy().astype(np.float64) - ref["scales"])) <= 1e-6
    if got2 is not None:
        assert np.array_equal(u32(got2["tile_mask"]), ref["tile_mask"])
        assert np.array_equal(u32(got2["hist"]), ref["hist"])


def test_quadtree_then_balance_on_cfg4(noit, cfg4_small):
    """S6 -> NEXT-1 chained on a resolved frame: masks from noit_quadtree, balanced in place."""
    sc = cfg4_small
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    fb = noit.DeviceFragBuf.from_host(sc.full)
    img = ctx.resolve(fb, BG)["final"]
    qt = ctx.quadtree(img, fb.width, fb.height, var_threshold_q=6)
    ref_qt = oracle.quadtree(img.cpu().numpy(), fb.width, fb.height, 0, 6)
    ref = oracle.quadtree_balance(ref_qt["tile_mask"], fb.width, fb.height)
    got = ctx.quadtree_balance(qt["tile_mask"], fb.width, fb.height)
    for k in ("tile_mask", "hist"):
        assert np.array_equal(u32(got[k]), ref[k]), k
    for k in ("tile_level", "cell_level"):
        assert np.array_equal(got[k].cpu().numpy(), ref[k]), k
    lv = ref["tile_level"].reshape((fb.height + 63) // 64, (fb.width + 63) // 64).astype(int)
    assert np.all(np.abs(np.diff(lv, axis=0)) <= 1) and np.all(np.abs(np.diff(lv, axis=1)) <= 1)
    assert np.max(np.abs(got["scales"].cpu().numpy() - ref["scales"])) <= 1e-6


@pytest.mark.parametrize("s2,s3", [(1.0, 1.0), (0.5, 0.5), (0.5, 0.25), (0.25, 0.25), (1.0, 0.25),
                                   (1.0, 0.5), (0.25, 0.5), (0.8, 0.36)])
def test_frame_global_pass_resolution(noit, cfg4_small, s2, s3):
    """O7g: pass 2 / pass 3 lods for the whole frame, snapped on the device from the scales."""
    sc = cfg4_small
    fb, hb, qb = (noit.DeviceFragBuf.from_host(b) for b in (sc.full, sc.half, sc.quarter))
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    scales = torch.tensor([2.0, s2, s3], dtype=torch.float32, device="cuda")
    got = ctx.resolve(fb, BG, half=hb, quarter=qb, pass_scales=scales)
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    ref = oracle.resolve_global(sc.full, sc.half, sc.quarter, w_eff, BG, oracle.snap_lod(s2),
                                oracle.snap_lod(s3))
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
    lay = oracle.build_features(sc.full)
    mag = mlp_magnitude(w_eff, np.maximum(lay["features"], [[64, 1, 1, 1, 1]]))
    extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
    for k in ("trans", "final"):
        close(got[k].cpu().numpy(), ref[k], extra=extra)
        assert np.max(np.abs(got[k].cpu().numpy()[:, :3] - ref[k][:, :3])) <= 2e-3


def test_frame_global_chain_from_device_scales(noit, cfg4_small):
    """quadtree -> balance (w, s_2, s_3 on the device) -> resolve at those pass resolutions, with
    no host round trip between the calls."""
    sc = cfg4_small
    fb, hb, qb = (noit.DeviceFragBuf.from_host(b) for b in (sc.full, sc.half, sc.quarter))
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    img = ctx.resolve(fb, BG)["final"]
    qt = ctx.quadtree(img, fb.width, fb.height, var_threshold_q=6)
    bal = ctx.quadtree_balance(qt["tile_mask"], fb.width, fb.height)
    got = ctx.resolve(fb, BG, half=hb, quarter=qb, pass_scales=bal["scales"])
    sc_host = bal["scales"].cpu().numpy()
    lod2, lod3 = oracle.snap_lod(sc_host[1]), oracle.snap_lod(sc_host[2])
    assert lod3 >= lod2                                                        # delta_3 > delta_2
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    ref = oracle.resolve_global(sc.full, sc.half, sc.quarter, w_eff, BG, lod2, lod3)
    lay = oracle.build_features(sc.full)
    mag = mlp_magnitude(w_eff, np.maximum(lay["features"], [[64, 1, 1, 1, 1]]))
    extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
    for k in ("trans", "final"):
        close(got[k].cpu().numpy(), ref[k], extra=extra)


# -------------------------------------------------------------------------------------------
# NEXT-2: temporal tile state (O11)
# -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,W,H,metric,step,hist_", [(0, 520, 330, 0, 1, True), (1, 520, 330, 1, 1, True),
                                                        (2, 1920, 1080, 0, 1, True), (3, 200, 136, 0, 0, True),
                                                        (4, 200, 136, 1, 2, True), (5, 64, 64, 0, 1, False)])
def test_quadtree_temporal_random(noit, seed, W, H, metric, step, hist_):
    from test_oracle_pins import _random_valid_masks
    rng = np.random.default_rng(100 + seed)
    Tx, Ty = (W + 63) // 64, (H + 63) // 64
    img = (rng.random((H * W, 4)) * rng.random((H * W, 1)) ** 3).astype(np.float32)
    yy = np.arange(H * W) // W
    img[yy < H // 3] = 0.25                                                    # a flat band: merges
    prev = _random_valid_masks(rng, Tx * Ty) if hist_ else None
    kw = dict(metric=metric, var_split=2500, var_merge=1500, corner_split=0.35, corner_merge=0.2,
              max_step=step)
    ref = oracle.quadtree_temporal(img, W, H, prev, **kw)
    ctx = noit.Noit()
    d_prev = None if prev is None else torch.from_numpy(prev.view(np.int32).copy()).cuda()
    got = ctx.quadtree_temporal(torch.from_numpy(img).cuda(), W, H, d_prev, **kw)
    qt_equal(got, ref)
    if prev is not None:
        assert not np.array_equal(ref["tile_mask"], oracle.quadtree_temporal(img, W, H, None, **kw)["tile_mask"])


@pytest.mark.parametrize("metric", [0, 1])
def test_quadtree_temporal_literal_threshold_order(noit, metric):
    """P:61's literal order (split threshold below the merge threshold) is callable and equals the
    oracle over a chain of frames; a node in the band alternates (pinned on the CPU)."""
    from test_oracle_pins import _random_valid_masks
    rng = np.random.default_rng(300 + metric)
    W, H = 333, 200
    Tx, Ty = (W + 63) // 64, (H + 63) // 64
    img = (rng.random((H * W, 4)) * rng.random((H * W, 1)) ** 3).astype(np.float32)
    d_img = torch.from_numpy(img).cuda()
    kw = dict(metric=metric, var_split=1500, var_merge=2500, corner_split=0.2, corner_merge=0.35, max_step=1)
    ctx = noit.Noit()
    r_prev = _random_valid_masks(rng, Tx * Ty)
    g_prev = torch.from_numpy(r_prev.view(np.int32).copy()).cuda()
    masks = []
    for _ in range(4):
        ref = oracle.quadtree_temporal(img, W, H, r_prev, **kw)
        got = ctx.quadtree_temporal(d_img, W, H, g_prev, **kw)
        qt_equal(got, ref)
        r_prev, g_prev = ref["tile_mask"], got["tile_mask"]
        masks.append(ref["tile_mask"].copy())
    assert len({m.tobytes() for m in masks}) >= 2              # the history matters over the chain


def test_quadtree_temporal_chain_over_cfg5_frames(noit):
    """Tiles of frame t steer frame t+1: four frames of the reduced cfg5 sequence."""
    seq = noit_scenes.cfg5(0, W=960, H=540)
    ctx = noit.Noit(seq.weights, seq.mlp_precision)
    W, H = seq.width, seq.height
    g_prev = r_prev = None
    depths = []
    for t in range(4):
        fb = noit.DeviceFragBuf.from_host(seq.frame(t))
        img = ctx.resolve(fb, seq.background, want=("final",))["final"]
        got = ctx.quadtree_temporal(img, W, H, g_prev, var_split=6, var_merge=3, max_step=1)
        ref = oracle.quadtree_temporal(img.cpu().numpy(), W, H, r_prev, var_split=6, var_merge=3, max_step=1)
        qt_equal(got, ref)
        g_prev, r_prev = got["tile_mask"], ref["tile_mask"]
        depths.append(ref["hist"].tolist())
    assert depths[0] != depths[1]                                              # the history matters


# -------------------------------------------------------------------------------------------
# NEXT-3: the paper's tile geometry, 16x16 -> 2x2
# -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,W,H,metric", [(0, 1920, 1080, 1), (1, 1920, 1080, 0), (2, 37, 21, 0),
                                             (3, 37, 21, 1), (4, 333, 130, 0), (5, 16, 16, 1)])
def test_quadtree16_random_images(noit, seed, W, H, metric):
    rng = np.random.default_rng(200 + seed)
    img = (rng.random((H * W, 4)) * rng.random((H * W, 1)) ** 2).astype(np.float32)
    yy = np.arange(H * W) // W
    img[yy < H // 3] = 0.4
    ref = oracle.quadtree16(img, W, H, metric, 900, 0.2)
    got = noit.Noit().quadtree16(torch.from_numpy(img).cuda(), W, H, metric, 900, 0.2)
    qt_equal(got, ref)
    assert len(set(ref["tile_mask"].tolist())) > 1 or W * H <= 256


def test_abi_errors(noit, cfg1_scene):
    import ctypes as C
    sc = cfg1_scene
    fb = noit.DeviceFragBuf.from_host(sc.full)
    ctx = noit.Noit()
    with pytest.raises(noit.NoitError) as e:
        ctx.resolve(fb, BG)
    assert e.value.status == 4                                   # NOIT_ERR_NO_WEIGHTS
    with pytest.raises(noit.NoitError) as e:
        ctx.set_weights(np.zeros(770, np.float32))
    assert e.value.status == 2
    with pytest.raises(noit.NoitError) as e:
        ctx.set_weights(sc.weights, 7)
    assert e.value.status == 3
    ctx.set_weights(sc.weights, 0)
    L = noit.lib()
    assert L.noit_resolve(None, None, None) == 1
    assert L.noit_resolve(ctx._ctx, None, None) == 1
    assert b"desc is NULL" in L.noit_last_error(ctx._ctx)
    launches = ctx.launch_count
    out = torch.full((fb.num_pixels, 4), 7.0, device="cuda")
    d = ctx.make_resolve_desc(fb, BG, out_final=out)
    d.full.width = 0
    assert L.noit_resolve(ctx._ctx, C.byref(d), None) == 2
    d = ctx.make_resolve_desc(fb, BG, out_final=out)
    d.full.color_fmt = 9
    assert L.noit_resolve(ctx._ctx, C.byref(d), None) == 3
    d = ctx.make_resolve_desc(fb, BG, out_final=out)
    d.out_final = out.data_ptr() + 4                             # misaligned
    assert L.noit_resolve(ctx._ctx, C.byref(d), None) == 3
    d = ctx.make_resolve_desc(fb, BG)
    assert L.noit_resolve(ctx._ctx, C.byref(d), None) == 1       # every output NULL
    torch.cuda.synchronize()
    assert ctx.launch_count == launches and torch.all(out == 7.0)   # nothing ran, outputs untouched
    with pytest.raises(noit.NoitError):
        ctx.quadtree(out, 0, 64)
    assert L.noit_infer(ctx._ctx, None, C.c_uint32(5), None, None) == 1
    assert L.noit_last_error(None) is not None


# -------------------------------------------------------------------------------------------
# the launch configuration bench.py times: the whole step as ONE CUDA graph with frame 3
# (reprojection + fallback, second context, side stream) forked beside frame 2 (quadtree +
# balance + adaptive resolve) after the plain resolve
# -------------------------------------------------------------------------------------------
def test_forked_graph_step_equals_the_eager_step_and_the_oracle(noit, cfg4_small):
    sc = cfg4_small
    W, H, P = sc.full.width, sc.full.height, sc.full.num_pixels
    fb, hb, qb = (noit.DeviceFragBuf.from_host(b) for b in (sc.full, sc.half, sc.quarter))
    ctx, ctx_b = noit.Noit(sc.weights, sc.mlp_precision), noit.Noit(sc.weights, sc.mlp_precision)
    M = np.eye(4, dtype=np.float32)
    M[0, 3] = 2.0 * 1.5 / W                                                    # 1.5-pixel camera shift
    f32 = dict(dtype=torch.float32, device="cuda")
    plain = dict(trans=torch.empty((P, 4), **f32), final=torch.empty((P, 4), **f32), depth1=torch.empty(P, **f32))
    adapt = dict(trans=torch.empty((P, 4), **f32), final=torch.empty((P, 4), **f32), depth1=torch.empty(P, **f32))
    st = dict(qt=None, bal=None, rp=None)
    side = torch.cuda.Stream()

    def frame3(c):
        st["rp"] = c.reproject(W, H, M, 1e-3, BG, plain["trans"], plain["depth1"], plain["depth1"], out=st["rp"])
        rp = st["rp"]
        c.resolve(fb, BG, want=(), out=dict(trans=rp["trans"], final=rp["final"], depth1=rp["depth"]),
                  pixel_list=rp["reject_list"], pixel_count=rp["reject_count"])

    def frame2():
        st["qt"] = ctx.quadtree(plain["final"], W, H, 0, 6, out=st["qt"])
        st["bal"] = ctx.quadtree_balance(st["qt"]["tile_mask"], W, H, out=st["bal"])
        ctx.resolve(fb, BG, want=(), out=adapt, half=hb, quarter=qb, cell_level=st["bal"]["cell_level"])

    def serial():
        ctx.resolve(fb, BG, want=(), out=plain)
        frame2()
        frame3(ctx)

    def forked():
        cur = torch.cuda.current_stream()
        ctx.resolve(fb, BG, want=(), out=plain)
        side.wait_stream(cur)
        with torch.cuda.stream(side):
            frame3(ctx_b)
        frame2()
        cur.wait_stream(side)

    serial()
    torch.cuda.synchronize()
    keys = lambda: (plain["final"], adapt["final"], adapt["depth1"], st["rp"]["final"], st["rp"]["trans"],
                    st["rp"]["accept"], st["bal"]["cell_level"], st["qt"]["tile_mask"])
    snap = [t.clone() for t in keys()]
    n_rej = int(st["rp"]["reject_count"].item())
    assert 0 < n_rej < P
    forked()                                                                   # eager once: allocations
    torch.cuda.synchronize()
    for t in keys():                                                           # the replay must rewrite them
        if t.dtype == torch.float32:
            t.zero_()
    graph = torch.cuda.CUDAGraph()
    capture_stream = torch.cuda.Stream()
    with torch.cuda.graph(graph, stream=capture_stream):
        forked()
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    for a, b in zip(snap, keys()):
        assert torch.equal(a, b)
    assert int(st["rp"]["reject_count"].item()) == n_rej
    # and the serial eager step is the oracle's step (frame 3 = accepted + re-resolved pixels)
    w_eff = oracle.effective_weights(sc.weights, sc.mlp_precision)
    r = oracle.resolve(sc.full, w_eff, BG)
    rp = oracle.reproject(W, H, M, 1e-3, BG, plain["trans"].cpu().numpy(), plain["depth1"].cpu().numpy(),
                          plain["depth1"].cpu().numpy())
    assert np.array_equal(rp["accept"], st["rp"]["accept"].cpu().numpy())
    assert np.array_equal(r["depth1"], plain["depth1"].cpu().numpy())
    out = dict(trans=rp["trans"], final=rp["final"], depth1=rp["depth"])
    oracle.resolve(sc.full, w_eff, BG, pixel_list=rp["reject_list"], out=out)
    close(st["rp"]["final"].cpu().numpy(), out["final"])



# -------------------------------------------------------------------------------------------
# the sharded path on one GPU -- a frame resolved band by band equals the whole frame
# -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("world", [2, 3, 8])
def test_sharded_resolve_and_quadtree_equal_the_whole_frame(noit, world):
    """Row bands from shard_rows (64-row aligned, fragment balanced), rebased CSR arrays from
    slice_rows, one resolve + quadtree per band, gather_rows: bit for bit the whole-frame result
    (every pixel and every 64x64 tile is independent: no exchange)."""
    from paper_2606_16747_b200.sharding import gather_rows, shard_rows, slice_rows
    sc = noit_scenes.cfg2(0)
    fbh = sc.full
    W, H = fbh.width, fbh.height
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    whole = ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG)
    qt_whole = ctx.quadtree(whole["final"], W, H, 0, 6)
    bands = shard_rows(fbh.offsets, W, H, world)
    assert bands[0][0] == 0 and bands[-1][1] == H and all(a[1] == b[0] for a, b in zip(bands, bands[1:]))
    parts = {k: [] for k in ("trans", "final", "depth1")}
    masks, cells, hist = [], [], np.zeros(4, np.int64)
    frags = []
    for (y0, y1) in bands:
        if y1 == y0:
            for k in parts:
                parts[k].append(np.zeros((0, 4) if k != "depth1" else (0,), np.float32))
            continue
        off, depth, rgba = slice_rows(fbh.offsets, fbh.depth, fbh.rgba, W, y0, y1)
        frags.append(int(off[-1]))
        band = FragBuf(W, y1 - y0, off, depth.copy(), rgba.copy())
        got = ctx.resolve(noit.DeviceFragBuf.from_host(band), BG)
        for k in parts:
            parts[k].append(got[k].cpu().numpy())
        q = ctx.quadtree(got["final"], W, y1 - y0, 0, 6)
        masks.append(u32(q["tile_mask"]))
        cells.append(q["cell_level"].cpu().numpy())
        hist += u32(q["hist"]).astype(np.int64)
    for k, ch in (("trans", 4), ("final", 4), ("depth1", 1)):
        assert np.array_equal(gather_rows(parts[k], bands, W, H, ch), whole[k].cpu().numpy()), k
    assert np.array_equal(np.concatenate(masks), u32(qt_whole["tile_mask"]))
    assert np.array_equal(np.concatenate(cells), qt_whole["cell_level"].cpu().numpy())
    assert np.array_equal(hist, u32(qt_whole["hist"]).astype(np.int64))
    if world == 2:
        assert abs(frags[0] - frags[1]) < 0.2 * sum(frags)       # balanced by fragments


@pytest.mark.parametrize("W,H,cuts", [(1920, 1080, (6, 11)), (3840, 2160, (1, 2, 20)), (640, 1000, (8,))])
def test_band_balance_with_a_mask_halo_equals_the_whole_frame(noit, W, H, cuts):
    """NEXT-1 across bands: each band balanced with its neighbours' nearest two tile
    rows of ORIGINAL masks (the halo exchange_halo_rows would move) equals the whole-frame 2:1
    balance bit for bit -- masks, tile levels, cell levels -- and the bands' histograms add up to
    the frame's.  Without the halo a band boundary may break the 2:1 rule (asserted too)."""
    from test_oracle_pins import _random_valid_masks
    from paper_2606_16747_b200.sharding import balance_band
    rng = np.random.default_rng(W + H)
    Tx, Ty = (W + 63) // 64, (H + 63) // 64
    m = _random_valid_masks(rng, Tx * Ty)
    ctx = noit.Noit()
    whole = ctx.quadtree_balance(torch.from_numpy(m.view(np.int32).copy()).cuda(), W, H)
    ref = oracle.quadtree_balance(m, W, H)
    assert np.array_equal(u32(whole["tile_mask"]), ref["tile_mask"])
    d = torch.from_numpy(m.view(np.int32).copy()).cuda().reshape(Ty, Tx)
    rows = [0, *cuts, Ty]
    hist = np.zeros(4, np.int64)
    differs_without_halo = False
    cw = (W + 7) // 8
    for r0, r1 in zip(rows[:-1], rows[1:]):
        y0, y1 = r0 * 64, min(H, r1 * 64)
        above = d[max(0, r0 - 2):r0].contiguous() if r0 > 0 else None
        below = d[r1:min(Ty, r1 + 2)].contiguous() if r1 < Ty else None
        got = balance_band(ctx, d[r0:r1].contiguous().reshape(-1), W, y0, y1, H, above, below)
        assert np.array_equal(u32(got["tile_mask"]), ref["tile_mask"][r0 * Tx:r1 * Tx])
        assert np.array_equal(got["tile_level"].cpu().numpy(), ref["tile_level"][r0 * Tx:r1 * Tx])
        c0, c1 = (y0 // 8) * cw, ((y1 + 7) // 8) * cw
        assert np.array_equal(got["cell_level"].cpu().numpy(), ref["cell_level"][c0:c1])
        hist += u32(got["hist"]).astype(np.int64)
        alone = balance_band(ctx, d[r0:r1].contiguous().reshape(-1), W, y0, y1, H)
        differs_without_halo |= not np.array_equal(u32(alone["tile_mask"]), ref["tile_mask"][r0 * Tx:r1 * Tx])
    assert np.array_equal(hist, ref["hist"].astype(np.int64))
    assert differs_without_halo or W < 1920                    # the halo is what makes the bands agree


def test_band_reprojection_with_a_row_halo(noit):
    """S8 across bands: a band extended by halo_rows(H) rows of its neighbours'
    prev_trans / prev_depth (here: slices of the whole previous frame stand in for the peer copies
    exchange_halo_rows makes), reprojected with band_matrix.  Bit-exact against the oracle on the
    band's inputs, and -- up to fp32 rounding at pixel edges / at the threshold -- the whole-frame
    reprojection restricted to the band: no pixel is rejected for want of a neighbour's row."""
    from paper_2606_16747_b200.sharding import band_matrix, extended_band, halo_rows, shard_rows
    seq = noit_scenes.cfg5(0, W=960, H=540)
    W, H = seq.width, seq.height
    ctx = noit.Noit(seq.weights, seq.mlp_precision)
    f0 = seq.frame(0)
    prev = ctx.resolve(noit.DeviceFragBuf.from_host(f0), seq.background)
    M = seq.reproject_matrix(1)
    whole = ctx.reproject(W, H, M, seq.depth_threshold, seq.background, prev["trans"], prev["depth1"],
                          prev["depth1"])
    acc_whole = whole["accept"].cpu().numpy().reshape(H, W)
    halo = halo_rows(H)
    p_t, p_d = prev["trans"].reshape(H, W, 4), prev["depth1"].reshape(H, W)
    for (y0, y1) in shard_rows(f0.offsets, W, H, 3):
        e0, e1 = extended_band((y0, y1), halo, H)
        He = e1 - e0
        Mb = band_matrix(M, H, e0, e1).astype(np.float32)
        bt = p_t[e0:e1].reshape(-1, 4).contiguous()
        bd = p_d[e0:e1].reshape(-1).contiguous()
        got = ctx.reproject(W, He, Mb, seq.depth_threshold, seq.background, bt, bd, bd)
        ref = oracle.reproject(W, He, Mb, seq.depth_threshold, seq.background, bt.cpu().numpy(),
                               bd.cpu().numpy(), bd.cpu().numpy())
        acc = got["accept"].cpu().numpy()
        assert np.array_equal(acc, ref["accept"])
        m = acc.astype(bool)
        assert np.array_equal(got["trans"].cpu().numpy()[m], ref["trans"][m])
        assert np.array_equal(got["depth"].cpu().numpy()[m], ref["depth"][m])
        own = acc.reshape(He, W)[y0 - e0:y1 - e0]
        differ = (own != acc_whole[y0:y1]).mean()
        assert differ < 2e-3, differ
        both = (own == 1) & (acc_whole[y0:y1] == 1)
        a = got["trans"].reshape(He, W, 4)[y0 - e0:y1 - e0].cpu().numpy()[both]
        b = whole["trans"].reshape(H, W, 4)[y0:y1].cpu().numpy()[both]
        assert (a == b).all(axis=1).mean() > 0.995


def test_validate_fragbuf_and_host_resolve_reject_a_malformed_csr(noit, cfg1_scene):
    """The hot kernels trust the CSR (documented precondition); noit_validate_fragbuf is the
    on-demand device check, and noit_resolve_host refuses a malformed CSR before it enqueues
    anything (outputs untouched)."""
    sc = cfg1_scene
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    fb = noit.DeviceFragBuf.from_host(sc.full)
    ctx.validate_fragbuf(fb)                                           # a good buffer passes
    for mutate in ("swap", "first", "last"):
        off = sc.full.offsets.copy()
        if mutate == "swap":
            k = int(np.argmax(np.diff(off.astype(np.int64)) > 0))
            off[k + 1] = off[k] - 1 if off[k] > 0 else off[k + 2] + 1   # decreasing step
            if off[k + 1] >= off[k] and off[k + 1] <= off[k + 2]:
                off[k + 1] = off[k + 2] + 5
        elif mutate == "first":
            off[0] = 1
        else:
            off[-1] += 3
        bad = noit.DeviceFragBuf(fb.width, fb.height, torch.from_numpy(off.view(np.int32)).cuda(), fb.depth, fb.rgba)
        with pytest.raises(noit.NoitError) as e:
            ctx.validate_fragbuf(bad)
        assert e.value.status == 3, mutate                              # NOIT_ERR_FORMAT
    # host entry point: band boundaries are checked before any copy is enqueued
    P = sc.full.num_pixels
    hb = FragBuf(sc.full.width, sc.full.height, sc.full.offsets.copy(), sc.full.depth, sc.full.rgba)
    hb.offsets[0] = 1                                                  # not a CSR: offsets[0] != 0
    final = np.full((P, 4), -1.0, np.float32)
    with pytest.raises(noit.NoitError) as e:
        ctx.resolve_host(hb, BG, out_final=final)
    assert e.value.status == 3 and (final == -1.0).all()


def test_bounds_checked_build_counts_no_violation(noit):
    """Our own memcheck (compute-sanitizer is closed on the GPU pool): libnoit_debug.so checks every
    stage range and fragment range the staged kernel touches; tests/debug_bounds_worker.py drives it
    through every staging regime against the oracle.  Zero violations, and the counter is shown to
    be live on a malformed CSR."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    dbg = os.path.join(root, "paper_2606_16747_b200", "libnoit_debug.so")
    if not os.path.exists(dbg):                               # a checkout that was never built: build it here
        from paper_2606_16747_b200 import _build
        _build.build(force=True)
    assert os.path.exists(dbg), "libnoit_debug.so missing: run __graft_entry__.build()"
    out = subprocess.run([sys.executable, os.path.join(root, "tests", "debug_bounds_worker.py")],
                         capture_output=True, text=True, timeout=900, env=dict(os.environ, NOIT_LIBRARY=dbg))
    assert out.returncode == 0, out.stderr[-3000:]
    rec = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert rec["cases"] >= 28 and rec["violations"] == 0, rec
    assert rec["fired_on_malformed_csr"] > 0, rec


def test_one_context_across_frame_sizes(noit):
    """Context scratch (G buffers, tile summary, balance scratch, counters) grows on demand and is
    kept between calls: one context driven through a small, a larger and again the small frame --
    plain, quadtree + balance, adaptive, reproject + pixel list -- must give exactly what fresh
    contexts give."""
    scenes = [noit_scenes.cfg4(1, W=192, H=136, n_prims=48, mean_band=(8.0, 10.0), cap=48),
              noit_scenes.cfg4(2, W=520, H=328, n_prims=96, mean_band=(10.0, 12.0), cap=64)]
    order = [0, 1, 0, 1]
    shared = noit.Noit(scenes[0].weights, scenes[0].mlp_precision)

    def run(ctx, sc):
        fb, hb, qb = (noit.DeviceFragBuf.from_host(b) for b in (sc.full, sc.half, sc.quarter))
        W, H = fb.width, fb.height
        plain = ctx.resolve(fb, BG)
        qt = ctx.quadtree(plain["final"], W, H, 0, 6)
        bal = ctx.quadtree_balance(qt["tile_mask"].clone(), W, H)
        ad = ctx.resolve(fb, BG, half=hb, quarter=qb, cell_level=bal["cell_level"])
        M = np.eye(4, dtype=np.float32)
        M[0, 3] = 2.0 * 2 / W
        rp = ctx.reproject(W, H, M, 1e-3, BG, plain["trans"], plain["depth1"], plain["depth1"])
        out = dict(trans=rp["trans"], final=rp["final"], depth1=rp["depth"])
        ctx.resolve(fb, BG, out=out, pixel_list=rp["reject_list"], pixel_count=rp["reject_count"])
        return [plain["final"], plain["trans"], qt["tile_mask"], bal["tile_mask"], bal["cell_level"], bal["hist"],
                ad["final"], rp["accept"], out["final"], out["trans"]]

    for k in order:
        sc = scenes[k]
        shared.set_weights(sc.weights, sc.mlp_precision)
        got = run(shared, sc)
        want = run(noit.Noit(sc.weights, sc.mlp_precision), sc)
        for i, (a, b) in enumerate(zip(got, want)):
            assert torch.equal(a, b), (k, i)
