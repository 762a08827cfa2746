"""GPU parity (`-m gpu`): the CUDA path through the C ABI versus the CPU oracle, element by
element on the same seeded inputs.  Classes:
  bit-exact  : idx1, idx2, count, depth1, tile_mask, cell_level, hist, accept, reject set,
               reprojected copies
  fp32       : |a-b| <= 1e-5 max(|a|,|b|) + 1e-6   (BASELINE.json north_star, as written:
               layers, tail accumulators, compositing, and the resolve's outputs)
  mlp guard  : + K_MLP * eps32 * T_2 * mag(f), K_MLP = 4, eps32 = 2^-24, mag(f) = the MLP evaluated
               with |W|, |b|, |x| (first-order forward bound of an fp32 evaluation in any order);
               at most 2.4e-7 * mag, where round 1 allowed 1e-5 * mag.  Measured on B200 it is never
               needed: the largest |a-b| / (1e-5 max + 1e-6) over cfg1-cfg3 and the random frames
               is 0.57 (printed per test in the terminal summary, tests/conftest.py).
  bf16 mode  : 2e-3 absolute on colour (north_star) on top of the bar above
"""
import numpy as np
import pytest
import torch

import noit_scenes
import oracle
from noit_scenes.raster import FragBuf

pytestmark = pytest.mark.gpu
BG = (0.2, 0.3, 0.4)


@pytest.fixture(scope="module")
def noit():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16747_b200 as m
    return m


K_MLP = 4.0
EPS32 = 2.0 ** -24
RATIOS = {}          # test id -> largest |a-b| / (1e-5 max(|a|,|b|) + 1e-6) seen (terminal summary)


def close(a, b, rel=1e-5, abs_=1e-6, extra=None):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    base = rel * np.maximum(np.abs(a), np.abs(b)) + abs_
    err = np.abs(a - b)
    if err.size:
        import os
        key = os.environ.get("PYTEST_CURRENT_TEST", "?").split(" ")[0].split("::")[-1]
        RATIOS[key] = max(RATIOS.get(key, 0.0), float((err / base).max()))
    tol = base if extra is None else base + extra
    bad = err > tol
    if bad.any():
        i = np.argwhere(bad)[0]
        raise AssertionError(f"{bad.sum()} mismatches, first at {tuple(i)}: {a[tuple(i)]} vs {b[tuple(i)]}")
    return True


def u32(t):
    return t.cpu().numpy().view(np.uint32)


def mlp_magnitude(w_eff, feats):
    """|W3|(|W2|(|W1||x|+|b1|)+|b2|)+|b3| in float64: scale of the rounding error of f(x)."""
    w = np.abs(w_eff.astype(np.float64))
    W1, b1 = w[:160].reshape(32, 5), w[160:192]
    W2, b2 = w[192:704].reshape(16, 32), w[704:720]
    W3, b3 = w[720:768].reshape(3, 16), w[768:771]
    x = np.abs(feats.astype(np.float64))
    return ((x @ W1.T + b1) @ W2.T + b2) @ W3.T + b3


def check_resolve(noit, fb_host, weights, precision, got, ref=None, bf16_abs=2e-3):
    w_eff = oracle.effective_weights(weights, precision)
    if ref is None:
        ref = oracle.resolve(fb_host, w_eff, BG)
    lay = oracle.build_features(fb_host)
    a1, a2 = lay["layer1"][:, 3].astype(np.float64), lay["layer2"][:, 3].astype(np.float64)
    t2 = (1 - a1) * (1 - a2)
    mag = mlp_magnitude(w_eff, lay["features"]) * t2[:, None]
    extra = np.concatenate([K_MLP * EPS32 * mag, np.zeros((mag.shape[0], 1))], axis=1)
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])          # bit-exact
    for k in ("trans", "final"):
        g = got[k].cpu().numpy()
        close(g, ref[k], extra=extra)
        if precision == 1:                       # BASELINE.json: 2e-3 absolute on colour
            assert np.max(np.abs(g[:, :3].astype(np.float64) - ref[k][:, :3])) <= bf16_abs
    return ref


def random_fb(rng, W, H, max_n, dtype, tie_frac=0.3, empty_frac=0.2, heavy=None):
    P = W * H
    counts = rng.integers(0, max_n + 1, P)
    counts[rng.random(P) < empty_frac] = 0
    if heavy:
        counts[rng.integers(0, P, heavy[0])] = heavy[1]
    off = np.zeros(P + 1, np.uint32)
    off[1:] = np.cumsum(counts)
    F = int(off[-1])
    depth = rng.uniform(0.01, 0.99, F).astype(np.float32)
    ties = rng.random(F) < tie_frac
    depth[ties] = rng.choice(np.asarray([0.25, 0.5, 0.75], np.float32), int(ties.sum()))
    rgba = rng.uniform(0, 1, (F, 4)).astype(dtype)
    return FragBuf(W, H, off, depth, rgba)


# -------------------------------------------------------------------------------------------
# S1-S3
# -------------------------------------------------------------------------------------------
def check_layers(noit, fb_host):
    ctx = noit.Noit()
    got = ctx.build_features(noit.DeviceFragBuf.from_host(fb_host))
    ref = oracle.build_features(fb_host)
    for k in ("idx1", "idx2", "count"):
        assert np.array_equal(u32(got[k]), ref[k]), k
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
    assert np.array_equal(got["layer1"].cpu().numpy(), ref["layer1"])          # exact copies
    assert np.array_equal(got["layer2"].cpu().numpy(), ref["layer2"])
    close(got["tail_raw"].cpu().numpy(), ref["tail_raw"])
    close(got["features"].cpu().numpy(), ref["features"])


def test_build_features_cfg1(noit, cfg1_scene):
    check_layers(noit, cfg1_scene.full)


@pytest.mark.parametrize("dtype,seed", [(np.float32, 1), (np.float16, 2)])
def test_build_features_random_ties(noit, dtype, seed):
    rng = np.random.default_rng(seed)
    check_layers(noit, random_fb(rng, 67, 45, 12, dtype, tie_frac=0.5))


def test_build_features_heavy_and_empty(noit):
    rng = np.random.default_rng(3)
    check_layers(noit, random_fb(rng, 50, 21, 6, np.float16, heavy=(20, 300)))
    empty = FragBuf(5, 3, np.zeros(16, np.uint32), np.zeros(0, np.float32), np.zeros((0, 4), np.float16))
    check_layers(noit, empty)


# -------------------------------------------------------------------------------------------
# S4
# -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [0, 1])
def test_infer(noit, precision):
    rng = np.random.default_rng(4)
    w = noit_scenes.mlp_weights(7)
    n = 10007
    x = np.concatenate([rng.integers(0, 129, (n, 1)).astype(np.float32),
                        rng.random((n, 4)).astype(np.float32)], axis=1)
    ctx = noit.Noit(w, precision)
    w_eff = oracle.effective_weights(w, precision)
    assert np.array_equal(ctx.get_weights(), w_eff)                  # same rounding, bit for bit
    got = ctx.infer(torch.from_numpy(x).cuda()).cpu().numpy()
    close(got, oracle.infer(w_eff, x), extra=K_MLP * EPS32 * mlp_magnitude(w_eff, x))
    assert ctx.infer(torch.empty((0, 5), device="cuda")).shape == (0, 3)


def test_infer_dfaoit_width(noit):
    """NEXT-4: the comparison system's 10 -> 32 -> 16 -> 3 sigmoid network (931 parameters)."""
    from test_oracle_pins import _weights931
    rng = np.random.default_rng(14)
    w = _weights931(5)
    n = 10007
    x = rng.random((n, 10)).astype(np.float32)
    x[:, 9] = rng.integers(0, 129, n)
    got = noit.Noit().infer_dfaoit(w, torch.from_numpy(x).cuda()).cpu().numpy()
    assert np.max(np.abs(got.astype(np.float64) - oracle.infer10(w, x))) <= 1e-5     # outputs in (0, 1)
    with pytest.raises(noit.NoitError):
        noit.Noit().infer_dfaoit(w[:771], torch.from_numpy(x).cuda())


@pytest.mark.parametrize("dtype,seed,shape,max_n,heavy", [
    (np.float16, 41, (130, 33), 40, (5, 700)), (np.float32, 42, (67, 45), 12, None),
    (np.float16, 43, (96, 5), 150, None), (np.float32, 44, (31, 7), 3, (2, 1500)), (np.float16, 45, (1, 1), 9, None)])
def test_resolve_dfaoit_random(noit, dtype, seed, shape, max_n, heavy):
    """NEXT-4 / O12: ten features built in the same scan (light, heavy and cold tiles), sigmoid
    network, Eq. 3 composite, against the oracle; features at the fp32 bar, colours (sigmoid
    outputs in (0,1)) at 1e-5 absolute on top of it, depth1 bit-exact."""
    from test_oracle_pins import _weights931
    rng = np.random.default_rng(seed)
    fbh = random_fb(rng, shape[0], shape[1], max_n, dtype, heavy=heavy)
    w = _weights931(seed)
    got = noit.Noit().resolve_dfaoit(noit.DeviceFragBuf.from_host(fbh), w, BG,
                                     want=("trans", "final", "depth1", "features10"))
    ref = oracle.resolve10(fbh, w, BG, want_features=True)
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
    close(got["features10"].cpu().numpy(), ref["features10"])
    for k in ("trans", "final"):
        close(got[k].cpu().numpy(), ref[k], extra=1e-5)
    n = np.diff(fbh.offsets.astype(np.int64))
    assert not got["trans"].cpu().numpy()[n == 0, :3].any()            # empty pixels: C_t = 0


def test_resolve_dfaoit_cfg3_full(noit, cfg3_scene):
    from test_oracle_pins import _weights931
    sc = cfg3_scene
    w = _weights931(3)
    ctx = noit.Noit()
    got = ctx.resolve_dfaoit(noit.DeviceFragBuf.from_host(sc.full), w, BG, want=("trans", "final", "depth1", "features10"))
    ref = oracle.resolve10(sc.full, w, BG, want_features=True)
    assert np.array_equal(got["depth1"].cpu().numpy(), ref["depth1"])
    close(got["features10"].cpu().numpy(), ref["features10"])
    for k in ("trans", "final"):
        close(got[k].cpu().numpy(), ref[k], extra=1e-5)
    with pytest.raises(noit.NoitError):
        ctx.resolve_dfaoit(noit.DeviceFragBuf.from_host(sc.full), w[:771], BG)


# -------------------------------------------------------------------------------------------
# S1-S5 fused
# -------------------------------------------------------------------------------------------
def test_resolve_cfg1(noit, cfg1_scene):
    sc = cfg1_scene
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    got = ctx.resolve(noit.DeviceFragBuf.from_host(sc.full), BG)
    check_resolve(noit, sc.full, sc.weights, sc.mlp_precision, got)


@pytest.mark.parametrize("dtype,precision,seed,shape", [
    (np.float32, 0, 11, (67, 45)), (np.float16, 1, 12, (130, 33)), (np.float16, 0, 13, (31, 7)),
    (np.float16, 1, 14, (1, 1)), (np.float32, 1, 15, (257, 3))])
def test_resolve_random_ragged(noit, dtype, precision, seed, shape):
    rng = np.random.default_rng(seed)
    fbh = random_fb(rng, shape[0], shape[1], 40, dtype, heavy=(5, 700))
    w = noit_scenes.mlp_weights(seed)
    ctx = noit.Noit(w, precision)
    got = ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG)
    check_resolve(noit, fbh, w, precision, got)


@pytest.mark.parametrize("dtype,lo,hi", [
    (np.float16, 100, 128), (np.float32, 100, 128), (np.float16, 180, 188), (np.float32, 150, 157),
    (np.float16, 60, 70), (np.float32, 36, 40), (np.float16, 28, 32)])
def test_resolve_dense_tiles(noit, dtype, lo, hi):
    """Every tile near a staging boundary of the staged kernel: whole-tile stage, depth-only
    chunks of 4 / 2 rounds, colour chunks of 2 / 1 rounds, rounds that barely fit or do not."""
    rng = np.random.default_rng(lo * 1000 + hi)
    W, H = 96, 5
    counts = rng.integers(lo, hi + 1, W * H)
    off = np.zeros(W * H + 1, np.uint32)
    off[1:] = np.cumsum(counts)
    F = int(off[-1])
    depth = rng.uniform(0.01, 0.99, F).astype(np.float32)
    ties = rng.random(F) < 0.2
    depth[ties] = rng.choice(np.asarray([0.125, 0.5], np.float32), int(ties.sum()))
    fbh = FragBuf(W, H, off, depth, rng.uniform(0, 1, (F, 4)).astype(dtype))
    w = noit_scenes.mlp_weights(7)
    ctx = noit.Noit(w, 1)
    got = ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG)
    check_resolve(noit, fbh, w, 1, got)


@pytest.mark.parametrize("block", range(4))
def test_resolve_random_stress(noit, block):
    """48 small random frames: odd sizes (P not a multiple of 32, F not a multiple of 4), every list
    length regime (empty .. far above the 128 cap: the cold global path), both colour formats and
    weight precisions, exact depth ties."""
    rng = np.random.default_rng(1000 + block)
    for _ in range(12):
        W, H = int(rng.integers(1, 90)), int(rng.integers(1, 30))
        max_n = int(rng.choice([1, 3, 12, 40, 130, 300]))
        dtype = np.float16 if rng.random() < 0.6 else np.float32
        precision = int(rng.integers(0, 2))
        heavy = (int(rng.integers(1, 6)), int(rng.choice([200, 700, 1700]))) if rng.random() < 0.4 else None
        fbh = random_fb(rng, W, H, max_n, dtype, tie_frac=float(rng.choice([0.0, 0.3, 0.9])),
                        empty_frac=float(rng.choice([0.0, 0.2, 0.7])), heavy=heavy)
        w = noit_scenes.mlp_weights(int(rng.integers(0, 1000)))
        ctx = noit.Noit(w, precision)
        got = ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG)
        check_resolve(noit, fbh, w, precision, got)


@pytest.mark.parametrize("dtype,precision", [(np.float16, 1), (np.float32, 0)])
def test_resolve_alpha_exactly_zero_and_one(noit, dtype, precision):
    """Degenerate opacities the method has: alpha exactly 1 in the tail gives
    T_tail = 0 while A_tail > 0; alpha exactly 0 everywhere in the tail gives A_tail = 0 with
    N > 2 (reading A2: has_tail false, tail term forced to 0, features (N, 1, 0, 0, 0)); whole
    pixels of alpha 0 or 1; light and heavy lists."""
    rng = np.random.default_rng(77 + precision)
    fbh = random_fb(rng, 130, 21, 24, dtype, tie_frac=0.2, empty_frac=0.05, heavy=(6, 400))
    off = fbh.offsets.astype(np.int64)
    n = np.diff(off)
    pix = np.repeat(np.arange(n.size), n)
    a = fbh.rgba[:, 3].astype(np.float32)
    u = rng.random(a.size)
    a[u < 0.25] = 0.0
    a[u > 0.75] = 1.0
    kind = rng.integers(0, 5, n.size)                       # per pixel: 0-1 mixed, 2 all zero, 3 all one,
    a[kind[pix] == 2] = 0.0                                 # 4 tail of zeros behind two opaque-ish layers
    a[kind[pix] == 3] = 1.0
    lay = oracle.build_features(fbh)
    k4 = np.nonzero((kind == 4) & (n > 2))[0]
    a[np.isin(pix, k4)] = 0.0
    for idx in ("idx1", "idx2"):
        a[off[k4] + lay[idx][k4].astype(np.int64)] = 0.5
    fbh.rgba[:, 3] = a.astype(dtype)
    lay = oracle.build_features(fbh)
    assert ((lay["tail_raw"][:, 3] == 0) & (n > 2)).sum() > 50          # all-zero tails with N > 2
    assert ((lay["tail_raw"][:, 4] == 0) & (lay["tail_raw"][:, 3] > 0)).sum() > 50   # T_tail = 0, A_tail > 0
    w = noit_scenes.mlp_weights(3)
    ctx = noit.Noit(w, precision)
    fb = noit.DeviceFragBuf.from_host(fbh)
    check_resolve(noit, fbh, w, precision, ctx.resolve(fb, BG))
    got = ctx.build_features(fb)
    assert np.array_equal(u32(got["idx1"]), lay["idx1"]) and np.array_equal(u32(got["idx2"]), lay["idx2"])
    close(got["features"].cpu().numpy(), lay["features"])
    close(got["tail_raw"].cpu().numpy(), lay["tail_raw"])
    # an all-zero tail is exactly the two-layer composite (north_star invariant, A2)
    z = (lay["tail_raw"][:, 3] == 0)
    final = ctx.resolve(fb, BG)["final"].cpu().numpy()
    close(final[z], oracle.exact(fbh, BG)["final"][z])


def test_resolve_per_pixel_background(noit):
    """NEXT-4: C_b varies over the image; the transparency result is unchanged."""
    rng = np.random.default_rng(33)
    fbh = random_fb(rng, 97, 31, 40, np.float16, heavy=(3, 300))
    w = noit_scenes.mlp_weights(4)
    ctx = noit.Noit(w, 1)
    bgi = rng.random((fbh.num_pixels, 4)).astype(np.float32)
    fb = noit.DeviceFragBuf.from_host(fbh)
    got = ctx.resolve(fb, (9.0, 9.0, 9.0), background_image=torch.from_numpy(bgi).cuda())
    ref = oracle.resolve(fbh, oracle.effective_weights(w, 1), (9.0, 9.0, 9.0), background_image=bgi)
    check_resolve(noit, fbh, w, 1, got, ref=ref)
    plain = ctx.resolve(fb, BG)
    assert torch.equal(plain["trans"], got["trans"])


def test_resolve_empty_and_single_output(noit):
    w = noit_scenes.mlp_weights(0)
    ctx = noit.Noit(w, 0)
    empty = FragBuf(40, 3, np.zeros(121, np.uint32), np.zeros(0, np.float32), np.zeros((0, 4), np.float16))
    got = ctx.resolve(noit.DeviceFragBuf.from_host(empty), BG)
    assert torch.all(got["trans"] == torch.tensor([0, 0, 0, 1.0], device="cuda"))
    assert torch.all(got["final"] == torch.tensor([BG[0], BG[1], BG[2], 0.0], device="cuda"))
    assert torch.all(got["depth1"] == 1.0)
    rng = np.random.default_rng(5)
    fbh = random_fb(rng, 64, 9, 10, np.float16)
    full = ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG)
    only = ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG, want=("final",))
    assert set(only) == {"final"} and torch.equal(only["final"], full["final"])


def test_resolve_empty_tail_is_exact_two_layer_composite(noit):
    """BASELINE.json invariant on the GPU path: n_p <= 2 => output == Eq. 1 on the fragments."""
    rng = np.random.default_rng(6)
    fbh = random_fb(rng, 96, 20, 2, np.float32, empty_frac=0.1)
    ctx = noit.Noit(noit_scenes.mlp_weights(1), 0)
    got = ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG)["final"].cpu().numpy()
    close(got, oracle.exact(fbh, BG)["final"])


@pytest.fixture(scope="module")
def cfg2_scene():
    return noit_scenes.cfg2(0)


@pytest.fixture(scope="module")
def cfg3_scene():
    return noit_scenes.cfg3(0)


def test_resolve_cfg2_full(noit, cfg2_scene):
    sc = cfg2_scene
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    got = ctx.resolve(noit.DeviceFragBuf.from_host(sc.full), BG)
    check_resolve(noit, sc.full, sc.weights, sc.mlp_precision, got)


def test_resolve_cfg3_full_and_layers(noit, cfg3_scene):
    """BASELINE.json's 1080p config at FULL size, element by element (the oracle needs ~1 s)."""
    sc = cfg3_scene
    fb = noit.DeviceFragBuf.from_host(sc.full)
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    got = ctx.resolve(fb, BG)
    check_resolve(noit, sc.full, sc.weights, sc.mlp_precision, got)
    lay = ctx.build_features(fb, want=("idx1", "idx2", "count"))
    ref = oracle.build_features(sc.full)
    for k in ("idx1", "idx2", "count"):
        assert np.array_equal(u32(lay[k]), ref[k]), k
    assert sc.meta["tie_pixels"] > 0.05 * sc.full.num_pixels


def test_resolve_is_repeatable_over_many_launches(noit, cfg2_scene, cfg3_scene):
    """Race / scheduling evidence without a race detector: tiles are dealt dynamically (four atomic
    ticket counters, re-armed by the last warp of each launch), so a lost or doubled ticket, a late
    counter add, or a race in a warp's stage would show up as an unwritten or differing pixel in
    SOME launch.  Every launch starts from outputs filled with NaN and must reproduce the first
    launch bit for bit: 60 launches of cfg2 (all light tiles), 25 of cfg3 (light, heavy, cold)."""
    for sc, n in ((cfg2_scene, 60), (cfg3_scene, 25)):
        fb = noit.DeviceFragBuf.from_host(sc.full)
        ctx = noit.Noit(sc.weights, sc.mlp_precision)
        P = sc.full.num_pixels
        out = dict(trans=torch.empty((P, 4), device="cuda"), final=torch.empty((P, 4), device="cuda"),
                   depth1=torch.empty(P, device="cuda"))
        d = ctx.make_resolve_desc(fb, BG, out["trans"], out["final"], out["depth1"])
        ref = None
        for i in range(n):
            for t in out.values():
                t.fill_(float("nan"))
            ctx.resolve_desc(d)
            if ref is None:
                ref = {k: v.clone() for k, v in out.items()}
                assert not any(torch.isnan(v).any().item() for v in ref.values())
            else:
                for k in out:
                    assert torch.equal(out[k], ref[k]), (sc.name, i, k)


def test_resolve_host_matches_device(noit, cfg1_scene):
    sc = cfg1_scene
    ctx = noit.Noit(sc.weights, sc.mlp_precision)
    dev = ctx.resolve(noit.DeviceFragBuf.from_host(sc.full), BG)
    P = sc.full.num_pixels
    trans, final, d1 = (np.zeros((P, 4), np.float32), np.zeros((P, 4), np.float32), np.zeros(P, np.float32))
    ctx.resolve_host(sc.full, BG, trans, final, d1)
    assert np.array_equal(trans, dev["trans"].cpu().numpy())
    assert np.array_equal(final, dev["final"].cpu().numpy())
    assert np.array_equal(d1, dev["depth1"].cpu().numpy())


def test_resolve_host_banded_matches_device(noit, cfg2_scene, cfg3_scene):
    """noit_resolve_host pipelines frames above 32 MB in bands of whole tiles over three streams
    (cfg2: 5 bands, cfg3: 8): every band boundary must give the same bits as the single launch,
    twice in a row on the same context (the staging area is reused), from pinned and from
    pageable host memory."""
    for sc in (cfg2_scene, cfg3_scene):
        ctx = noit.Noit(sc.weights, sc.mlp_precision)
        dev = ctx.resolve(noit.DeviceFragBuf.from_host(sc.full), BG)
        P = sc.full.num_pixels
        for pinned in (False, True, True):
            mk = (lambda *sh: torch.zeros(sh, dtype=torch.float32).pin_memory()) if pinned else \
                (lambda *sh: np.zeros(sh, np.float32))
            trans, final, d1 = mk(P, 4), mk(P, 4), mk(P)
            ctx.resolve_host(sc.full, BG, trans, final, d1)
            for got, want in ((trans, dev["trans"]), (final, dev["final"]), (d1, dev["depth1"])):
                got = got.numpy() if pinned else got
                assert np.array_equal(got, want.cpu().numpy())

