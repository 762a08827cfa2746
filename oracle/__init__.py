"""ctypes loader for the CPU oracle (oracle/noit_oracle.c).

TEST INFRASTRUCTURE ONLY: may be imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` legs, never by the product package.  It does not import the
product package and shares no code with it.  Arguments are numpy arrays (host memory); this
file only marshals them -- all arithmetic is in noit_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "noit_oracle.c")
_LIB = os.path.join(_HERE, "libnoit_oracle.so")
ABSENT = 0xFFFFFFFF
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _chk(a, dtype, n=None):
    assert a.dtype == dtype and a.flags["C_CONTIGUOUS"], (a.dtype, dtype)
    if n is not None:
        assert a.size == n, (a.size, n)
    return a


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def effective_weights(weights: np.ndarray, precision: int) -> np.ndarray:
    """fp32 weights as given (0) or each rounded to bf16 RNE and widened (1)."""
    w = np.ascontiguousarray(weights, np.float32).copy()
    if precision == 1:
        lib().oracle_round_weights_bf16(_p(w), C.c_int32(w.size))
    return w


def infer(weights_eff: np.ndarray, features: np.ndarray) -> np.ndarray:
    f = np.ascontiguousarray(features, np.float32)
    n = f.shape[0]
    out = np.empty((n, 3), np.float32)
    rc = lib().oracle_infer(_p(_chk(weights_eff, np.float32, 771)), _p(f), C.c_uint32(n), _p(out))
    assert rc == 0
    return out


def infer10(weights931: np.ndarray, features: np.ndarray) -> np.ndarray:
    """The 10-feature, sigmoid-output network DFAOIT uses (931 parameters; comparison variant)."""
    f = np.ascontiguousarray(features, np.float32)
    n = f.shape[0]
    assert f.shape[1] == 10
    out = np.empty((n, 3), np.float32)
    rc = lib().oracle_infer10(_p(_chk(weights931, np.float32, 931)), _p(f), C.c_uint32(n), _p(out))
    assert rc == 0
    return out


def _fb_args(fb):
    if fb is None:
        return [C.c_int32(0), C.c_int32(0), None, None, None]
    P = fb.width * fb.height
    _chk(fb.offsets, np.uint32, P + 1)
    _chk(fb.depth, np.float32)
    assert fb.rgba.dtype in (np.float16, np.float32) and fb.rgba.flags["C_CONTIGUOUS"]
    return [C.c_int32(fb.width), C.c_int32(fb.height), _p(fb.offsets), _p(fb.depth), _p(fb.rgba)]


def build_features(fb) -> dict:
    P = fb.width * fb.height
    out = dict(idx1=np.empty(P, np.uint32), idx2=np.empty(P, np.uint32),
               count=np.empty(P, np.uint32), layer1=np.empty((P, 4), np.float32),
               layer2=np.empty((P, 4), np.float32), depth1=np.empty(P, np.float32),
               tail_raw=np.empty((P, 5), np.float32), features=np.empty((P, 5), np.float32))
    rc = lib().oracle_build_features(*_fb_args(fb), C.c_int32(fb.color_fmt),
                                     *[_p(out[k]) for k in ("idx1", "idx2", "count", "layer1",
                                                            "layer2", "depth1", "tail_raw",
                                                            "features")])
    assert rc == 0
    return out


def resolve(fb, weights_eff, background, half=None, quarter=None, cell_level=None,
            level_to_lod=(2, 1, 0, 0), pixel_list=None, tail_override=None, out=None,
            background_image=None) -> dict:
    """S1-S5 (+S7 with cell_level, +S9 with pixel_list).  `out` lets S9 write into existing
    arrays (pixels not in the list stay untouched)."""
    P = fb.width * fb.height
    if out is None:
        out = dict(trans=np.zeros((P, 4), np.float32), final=np.zeros((P, 4), np.float32),
                   depth1=np.zeros(P, np.float32))
    bg = np.asarray(background, np.float32)
    l2l = np.asarray(level_to_lod, np.uint8)
    args = _fb_args(fb) + [C.c_int32(fb.color_fmt)]
    args += _fb_args(half) + _fb_args(quarter)
    if cell_level is not None:
        _chk(cell_level, np.uint8, ((fb.width + 7) // 8) * ((fb.height + 7) // 8))
    if pixel_list is not None:
        pixel_list = np.ascontiguousarray(pixel_list, np.uint32)
    if tail_override is not None:
        tail_override = np.ascontiguousarray(tail_override, np.float32)
        assert tail_override.size == 3 * P
    args += [_p(cell_level), _p(l2l),
             _p(None if weights_eff is None else _chk(weights_eff, np.float32, 771)),
             _p(tail_override), _p(bg), _p(pixel_list),
             C.c_uint32(0 if pixel_list is None else pixel_list.size),
             _p(out["trans"]), _p(out["final"]), _p(out["depth1"]),
             _p(None if background_image is None else _chk(np.ascontiguousarray(background_image, np.float32),
                                                           np.float32, 4 * P))]
    rc = lib().oracle_resolve(*args)
    assert rc == 0, rc
    return out


def snap_lod(scale) -> int:
    """Reading A27: power-of-two snap of an Eq. 2 scale (fp32 compare): 0 = full, 1 = half,
    2 = quarter resolution."""
    s = np.float32(scale)
    return 0 if s > np.float32(0.70710678) else (1 if s > np.float32(0.35355339) else 2)


def resolve_global(fb, half, quarter, weights_eff, background, lod2: int, lod3: int) -> dict:
    """O7g: layer 1 at full resolution, pass 2 (layer 2) at lod2 and pass 3 (tail) at lod3 for the
    whole frame, bilinear upsampling, features / MLP / composite at full resolution."""
    P = fb.width * fb.height
    out = dict(trans=np.zeros((P, 4), np.float32), final=np.zeros((P, 4), np.float32),
               depth1=np.zeros(P, np.float32))
    bg = np.asarray(background, np.float32)
    args = _fb_args(fb) + [C.c_int32(fb.color_fmt)] + _fb_args(half) + _fb_args(quarter)
    args += [C.c_int32(lod2), C.c_int32(lod3), _p(_chk(weights_eff, np.float32, 771)), _p(bg),
             _p(out["trans"]), _p(out["final"]), _p(out["depth1"])]
    rc = lib().oracle_resolve_global(*args)
    assert rc == 0, rc
    return out


def resolve10(fb, weights931, background, want_features: bool = False) -> dict:
    """O12 (NEXT-4): the DFAOIT resolve -- ten features from the fragment list, the 931-parameter
    sigmoid network predicting the whole transparency colour, Eq. 3 composite."""
    P = fb.width * fb.height
    out = dict(trans=np.zeros((P, 4), np.float32), final=np.zeros((P, 4), np.float32),
               depth1=np.zeros(P, np.float32))
    if want_features:
        out["features10"] = np.zeros((P, 10), np.float32)
    bg = np.asarray(background, np.float32)
    w = _chk(np.ascontiguousarray(weights931, np.float32), np.float32, 931)
    args = _fb_args(fb) + [C.c_int32(fb.color_fmt), _p(w), _p(bg), _p(out["trans"]), _p(out["final"]),
                           _p(out["depth1"]), _p(out.get("features10"))]
    rc = lib().oracle_resolve10(*args)
    assert rc == 0, rc
    return out


def exact(fb, background) -> dict:
    """O5x: full sort + Porter-Duff over (Eq. 1) + background; and the exact tail composite."""
    P = fb.width * fb.height
    bg = np.asarray(background, np.float32)
    final = np.empty((P, 4), np.float32)
    tail = np.empty((P, 3), np.float32)
    rc = lib().oracle_exact(*_fb_args(fb), C.c_int32(fb.color_fmt), _p(bg), _p(final), _p(tail))
    assert rc == 0
    return dict(final=final, tail=tail)


def quadtree(image: np.ndarray, width: int, height: int, metric: int = 0,
             var_threshold_q: int = 6, corner_threshold: float = 0.02) -> dict:
    img = _chk(np.ascontiguousarray(image, np.float32), np.float32, width * height * 4)
    Tx, Ty = (width + 63) // 64, (height + 63) // 64
    cx, cy = (width + 7) // 8, (height + 7) // 8
    out = dict(tile_mask=np.zeros(Tx * Ty, np.uint32), cell_level=np.zeros(cx * cy, np.uint8),
               hist=np.zeros(4, np.uint32))
    rc = lib().oracle_quadtree(_p(img), C.c_int32(width), C.c_int32(height), C.c_int32(metric),
                               C.c_uint32(var_threshold_q), C.c_float(corner_threshold),
                               _p(out["tile_mask"]), _p(out["cell_level"]), _p(out["hist"]))
    assert rc == 0
    return out


def quadtree16(image: np.ndarray, width: int, height: int, metric: int = 1,
               var_threshold_q: int = 6, corner_threshold: float = 0.02) -> dict:
    """O6 in the paper's own geometry: 16x16 base tiles down to 2x2 leaves."""
    img = _chk(np.ascontiguousarray(image, np.float32), np.float32, width * height * 4)
    Tx, Ty = (width + 15) // 16, (height + 15) // 16
    cx, cy = (width + 1) // 2, (height + 1) // 2
    out = dict(tile_mask=np.zeros(Tx * Ty, np.uint32), cell_level=np.zeros(cx * cy, np.uint8),
               hist=np.zeros(4, np.uint32))
    rc = lib().oracle_quadtree_base(_p(img), C.c_int32(width), C.c_int32(height), C.c_int32(metric),
                                    C.c_uint32(var_threshold_q), C.c_float(corner_threshold),
                                    C.c_int32(16), _p(out["tile_mask"]), _p(out["cell_level"]),
                                    _p(out["hist"]))
    assert rc == 0
    return out


def quadtree_balance(tile_mask: np.ndarray, width: int, height: int, iterations: int = 2,
                     delta2: float = 2.2, delta3: float = 3.0) -> dict:
    """O10: 2:1 tile balance by Jacobi relaxation + histogram + demand index and Eq. 2 scales."""
    Tx, Ty = (width + 63) // 64, (height + 63) // 64
    cx, cy = (width + 7) // 8, (height + 7) // 8
    out = dict(tile_mask=_chk(np.array(tile_mask, np.uint32), np.uint32, Tx * Ty),
               tile_level=np.zeros(Tx * Ty, np.uint8), cell_level=np.zeros(cx * cy, np.uint8),
               hist=np.zeros(4, np.uint32), scales=np.zeros(3, np.float32))
    rc = lib().oracle_quadtree_balance(C.c_int32(width), C.c_int32(height), C.c_int32(iterations),
                                       C.c_float(delta2), C.c_float(delta3), _p(out["tile_mask"]),
                                       _p(out["tile_level"]), _p(out["cell_level"]), _p(out["hist"]),
                                       _p(out["scales"]))
    assert rc == 0
    return out


def quadtree_temporal(image: np.ndarray, width: int, height: int, prev_mask=None, metric: int = 0,
                      var_split: int = 6, var_merge: int = 3, corner_split: float = 0.02,
                      corner_merge: float = 0.01, max_step: int = 1) -> dict:
    """O11: quadtree with split / merge hysteresis against the previous frame's masks and at most
    `max_step` levels of change per base tile and frame."""
    img = _chk(np.ascontiguousarray(image, np.float32), np.float32, width * height * 4)
    Tx, Ty = (width + 63) // 64, (height + 63) // 64
    cx, cy = (width + 7) // 8, (height + 7) // 8
    prev = None if prev_mask is None else _chk(np.ascontiguousarray(prev_mask, np.uint32), np.uint32, Tx * Ty)
    out = dict(tile_mask=np.zeros(Tx * Ty, np.uint32), cell_level=np.zeros(cx * cy, np.uint8),
               hist=np.zeros(4, np.uint32))
    rc = lib().oracle_quadtree_temporal(_p(img), C.c_int32(width), C.c_int32(height), C.c_int32(metric),
                                        C.c_uint32(var_split), C.c_uint32(var_merge),
                                        C.c_float(corner_split), C.c_float(corner_merge),
                                        C.c_int32(max_step), None if prev is None else _p(prev),
                                        _p(out["tile_mask"]), _p(out["cell_level"]), _p(out["hist"]))
    assert rc == 0
    return out


def reproject(width, height, M, depth_threshold, background, prev_trans, prev_depth, cur_depth,
              out_trans=None, out_depth=None, out_final=None) -> dict:
    P = width * height
    M = _chk(np.ascontiguousarray(M, np.float32).reshape(-1), np.float32, 16)
    bg = np.asarray(background, np.float32)
    out = dict(trans=np.zeros((P, 4), np.float32) if out_trans is None else out_trans,
               depth=np.zeros(P, np.float32) if out_depth is None else out_depth,
               final=np.zeros((P, 4), np.float32) if out_final is None else out_final,
               accept=np.zeros(P, np.uint8), reject_list=np.zeros(P, np.uint32))
    cnt = C.c_uint32(0)
    rc = lib().oracle_reproject(C.c_int32(width), C.c_int32(height), _p(M),
                                C.c_float(depth_threshold), _p(bg),
                                _p(_chk(prev_trans, np.float32, 4 * P)),
                                _p(_chk(prev_depth, np.float32, P)),
                                _p(_chk(cur_depth, np.float32, P)), _p(out["trans"]),
                                _p(out["depth"]), _p(out["final"]), _p(out["accept"]),
                                _p(out["reject_list"]), C.byref(cnt))
    assert rc == 0
    out["reject_count"] = int(cnt.value)
    out["reject_list"] = out["reject_list"][:cnt.value].copy()
    return out


def reproject_bilinear(width, height, M, depth_threshold, background, prev_trans, prev_depth,
                       cur_depth, out_trans=None, out_depth=None, out_final=None) -> dict:
    """O8b (A28): O8 with a bilinear fetch of the previous result where all four taps pass the
    disocclusion test; `filtered` marks those pixels."""
    P = width * height
    M = _chk(np.ascontiguousarray(M, np.float32).reshape(-1), np.float32, 16)
    bg = np.asarray(background, np.float32)
    out = dict(trans=np.zeros((P, 4), np.float32) if out_trans is None else out_trans,
               depth=np.zeros(P, np.float32) if out_depth is None else out_depth,
               final=np.zeros((P, 4), np.float32) if out_final is None else out_final,
               accept=np.zeros(P, np.uint8), reject_list=np.zeros(P, np.uint32),
               filtered=np.zeros(P, np.uint8))
    cnt = C.c_uint32(0)
    rc = lib().oracle_reproject_bilinear(C.c_int32(width), C.c_int32(height), _p(M),
                                         C.c_float(depth_threshold), _p(bg),
                                         _p(_chk(prev_trans, np.float32, 4 * P)),
                                         _p(_chk(prev_depth, np.float32, P)),
                                         _p(_chk(cur_depth, np.float32, P)), _p(out["trans"]),
                                         _p(out["depth"]), _p(out["final"]), _p(out["accept"]),
                                         _p(out["reject_list"]), C.byref(cnt), _p(out["filtered"]))
    assert rc == 0
    out["reject_count"] = int(cnt.value)
    out["reject_list"] = out["reject_list"][:cnt.value].copy()
    return out
