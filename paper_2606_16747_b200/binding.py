"""Thin ctypes binding over libnoit.so (include/noit.h).  Argument marshalling only: every
step of the path runs in the CUDA kernels behind the C ABI.  torch is used for device memory
and streams.  There is no CPU fallback: a missing library raises at import of this module's
`lib()`; nothing here imports or calls oracle/.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import _build

ABSENT = 0xFFFFFFFF
MLP_PARAMS = 771
RGBA_F16, RGBA_F32 = 0, 1
MLP_FP32, MLP_BF16 = 0, 1
QT_VARIANCE, QT_CORNER = 0, 1
STATUS = {0: "NOIT_OK", 1: "NOIT_ERR_NULL", 2: "NOIT_ERR_SIZE", 3: "NOIT_ERR_FORMAT",
          4: "NOIT_ERR_NO_WEIGHTS", 5: "NOIT_ERR_CUDA", 6: "NOIT_ERR_UNSUPPORTED"}
EXPORTS = ["noit_create", "noit_destroy", "noit_set_weights", "noit_get_weights",
           "noit_last_error", "noit_launch_count", "noit_build_features", "noit_infer",
           "noit_resolve", "noit_resolve_host", "noit_quadtree", "noit_quadtree_temporal",
           "noit_quadtree_balance", "noit_quadtree_balance_static", "noit_quadtree16", "noit_infer_dfaoit", "noit_resolve_dfaoit",
           "noit_validate_fragbuf", "noit_debug_bounds_violations",
           "noit_reproject"]


class NoitError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class FragBufC(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("num_fragments", C.c_uint32),
                ("color_fmt", C.c_int32), ("offsets", C.c_void_p), ("depth", C.c_void_p),
                ("rgba", C.c_void_p)]


class LayersC(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("idx1", "idx2", "count", "layer1", "layer2", "depth1",
                                          "tail_raw", "features")]


class ResolveDescC(C.Structure):
    _fields_ = [("full", FragBufC), ("half", C.POINTER(FragBufC)), ("quarter", C.POINTER(FragBufC)),
                ("cell_level", C.c_void_p), ("level_to_lod", C.c_uint8 * 4),
                ("background", C.c_float * 3), ("pixel_list", C.c_void_p),
                ("pixel_count", C.c_void_p), ("out_trans", C.c_void_p), ("out_final", C.c_void_p),
                ("out_depth1", C.c_void_p), ("pass_scales", C.c_void_p),
                ("background_image", C.c_void_p)]


class QtParamsC(C.Structure):
    _fields_ = [("metric", C.c_int32), ("var_threshold_q", C.c_uint32),
                ("corner_threshold", C.c_float)]


class QtTemporalParamsC(C.Structure):
    _fields_ = [("metric", C.c_int32), ("var_split_q", C.c_uint32), ("var_merge_q", C.c_uint32),
                ("corner_split", C.c_float), ("corner_merge", C.c_float), ("max_level_step", C.c_int32)]


class ReprojectDescC(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("M", C.c_float * 16),
                ("depth_threshold", C.c_float), ("background", C.c_float * 3),
                ("prev_trans", C.c_void_p), ("prev_depth", C.c_void_p), ("cur_depth", C.c_void_p),
                ("out_trans", C.c_void_p), ("out_depth", C.c_void_p), ("out_final", C.c_void_p),
                ("accept", C.c_void_p), ("reject_list", C.c_void_p), ("reject_count", C.c_void_p),
                ("filter", C.c_int32)]


_lib = None


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load libnoit.so (building it first if nvcc is here and the sources are newer)."""
    global _lib
    if _lib is None:
        path = os.environ.get("NOIT_LIBRARY") or _build.LIB      # NOIT_LIBRARY: another build of libnoit
        if path == _build.LIB and (not os.path.exists(path) or os.environ.get("NOIT_REBUILD")):
            path = _build.build()
        L = C.CDLL(path)
        L.noit_last_error.restype = C.c_char_p
        L.noit_launch_count.restype = C.c_uint64
        for name in EXPORTS:
            getattr(L, name)                      # raises AttributeError if a symbol is missing
        _lib = L
    return _lib


def _ptr(t):
    """Device pointer of a tensor (None stays NULL); a tensor on another device than the current one
    would be dereferenced by a context of the wrong device: refuse it here."""
    if t is None:
        return None
    if t.is_cuda and t.device.index != torch.cuda.current_device():
        raise ValueError(f"tensor on cuda:{t.device.index} passed while cuda:{torch.cuda.current_device()} is current")
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class DeviceFragBuf:
    """A CSR fragment buffer resident in HBM."""

    def __init__(self, width, height, offsets, depth, rgba):
        assert offsets.dtype == torch.int32 or offsets.dtype == torch.uint32
        assert depth.dtype == torch.float32 and rgba.dtype in (torch.float16, torch.float32)
        self.width, self.height = int(width), int(height)
        self.offsets, self.depth, self.rgba = offsets, depth, rgba
        self.num_fragments = int(depth.numel())
        self.color_fmt = RGBA_F16 if rgba.dtype == torch.float16 else RGBA_F32

    @staticmethod
    def from_host(fb, device="cuda") -> "DeviceFragBuf":
        """Upload a noit_scenes.FragBuf (numpy) byte for byte."""
        import numpy as np
        off = torch.from_numpy(fb.offsets.view(np.int32)).to(device)
        return DeviceFragBuf(fb.width, fb.height, off, torch.from_numpy(fb.depth).to(device),
                             torch.from_numpy(fb.rgba).to(device))

    @property
    def num_pixels(self):
        return self.width * self.height

    def c_struct(self) -> FragBufC:
        return FragBufC(self.width, self.height, self.num_fragments, self.color_fmt,
                        self.offsets.data_ptr(), self.depth.data_ptr() if self.num_fragments else 0,
                        self.rgba.data_ptr() if self.num_fragments else 0)

    def nbytes(self) -> int:
        return (self.offsets.numel() * 4 + self.depth.numel() * 4
                + self.rgba.numel() * self.rgba.element_size())


class Noit:
    """One libnoit context (weights + small device scratch).  Methods mirror the C entry points
    and enqueue on torch's current stream (or `stream`); outputs are torch tensors."""

    def __init__(self, weights=None, precision: int = MLP_FP32):
        self._L = lib()
        self._ctx = C.c_void_p()
        st = self._L.noit_create(C.byref(self._ctx))
        if st != 0:
            raise NoitError(st, self._L.noit_last_error(None).decode())
        if weights is not None:
            self.set_weights(weights, precision)

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self._L.noit_destroy(self._ctx)
            self._ctx = C.c_void_p()

    __del__ = close

    def _check(self, st: int):
        if st != 0:
            raise NoitError(st, self._L.noit_last_error(self._ctx).decode())

    # ---- context ----------------------------------------------------------------------
    def set_weights(self, weights, precision: int = MLP_FP32):
        import numpy as np
        w = np.ascontiguousarray(weights, np.float32)
        self._check(self._L.noit_set_weights(self._ctx, w.ctypes.data_as(C.c_void_p),
                                             C.c_int32(w.size), C.c_int32(precision)))

    def get_weights(self):
        import numpy as np
        w = np.empty(MLP_PARAMS, np.float32)
        self._check(self._L.noit_get_weights(self._ctx, w.ctypes.data_as(C.c_void_p),
                                             C.c_int32(MLP_PARAMS)))
        return w

    def debug_bounds_violations(self) -> int:
        """Violations counted by a NOIT_DEBUG_BOUNDS build of the library (0 in the release build)."""
        n = C.c_uint32(0)
        self._check(self._L.noit_debug_bounds_violations(self._ctx, C.byref(n)))
        return int(n.value)

    @property
    def launch_count(self) -> int:
        return int(self._L.noit_launch_count(self._ctx))

    def validate_fragbuf(self, fb: "DeviceFragBuf", stream=None):
        """Raises NoitError(NOIT_ERR_FORMAT) unless offsets are a CSR of fb.num_fragments fragments."""
        assert fb.offsets.device.index == torch.cuda.current_device(), "fragment buffer on another device"
        fbc = fb.c_struct()
        self._check(self._L.noit_validate_fragbuf(self._ctx, C.byref(fbc), _stream(stream)))

    # ---- S1-S3 ------------------------------------------------------------------------
    def build_features(self, fb: DeviceFragBuf, want=("idx1", "idx2", "count", "layer1", "layer2",
                                                      "depth1", "tail_raw", "features"), stream=None):
        P, dev = fb.num_pixels, fb.offsets.device
        shapes = dict(idx1=((P,), torch.int32), idx2=((P,), torch.int32), count=((P,), torch.int32),
                      layer1=((P, 4), torch.float32), layer2=((P, 4), torch.float32),
                      depth1=((P,), torch.float32), tail_raw=((P, 5), torch.float32),
                      features=((P, 5), torch.float32))
        out = {k: torch.empty(shapes[k][0], dtype=shapes[k][1], device=dev) for k in want}
        lay = LayersC(*[out[k].data_ptr() if k in out else None for k, _ in LayersC._fields_])
        fbc = fb.c_struct()
        self._check(self._L.noit_build_features(self._ctx, C.byref(fbc), C.byref(lay), _stream(stream)))
        return out

    # ---- S4 ---------------------------------------------------------------------------
    def infer(self, features: torch.Tensor, out=None, stream=None) -> torch.Tensor:
        assert features.dtype == torch.float32 and features.is_contiguous()
        n = features.shape[0]
        if out is None:
            out = torch.empty((n, 3), dtype=torch.float32, device=features.device)
        self._check(self._L.noit_infer(self._ctx, _ptr(features), C.c_uint32(n), _ptr(out),
                                       _stream(stream)))
        return out

    # ---- NEXT-4 (comparison variant) ------------------------------------------------------
    def infer_dfaoit(self, weights931, features: torch.Tensor, out=None, stream=None) -> torch.Tensor:
        """10-feature / sigmoid-output network (931 host parameters) on [n, 10] device features."""
        import numpy as np
        w = np.ascontiguousarray(weights931, np.float32)
        assert features.dtype == torch.float32 and features.is_contiguous()
        n = features.shape[0]
        if out is None:
            out = torch.empty((n, 3), dtype=torch.float32, device=features.device)
        self._check(self._L.noit_infer_dfaoit(self._ctx, w.ctypes.data_as(C.c_void_p), C.c_int32(w.size),
                                              _ptr(features), C.c_uint32(n), _ptr(out), _stream(stream)))
        return out

    def resolve_dfaoit(self, fb: "DeviceFragBuf", weights931, background=(0.0, 0.0, 0.0),
                       want=("trans", "final", "depth1"), out=None, stream=None):
        """NEXT-4 (O12): the DFAOIT resolve (ten features, Eq. 3).  `want` may include "features10"."""
        import numpy as np
        w = np.ascontiguousarray(weights931, np.float32)
        P, dev = fb.num_pixels, fb.offsets.device
        out = dict(out) if out else {}
        shapes = dict(trans=(P, 4), final=(P, 4), depth1=(P,), features10=(P, 10))
        for k in want:
            if k not in out:
                out[k] = torch.empty(shapes[k], dtype=torch.float32, device=dev)
        fbc = fb.c_struct()
        bg = (C.c_float * 3)(*background)
        self._check(self._L.noit_resolve_dfaoit(
            self._ctx, C.byref(fbc), w.ctypes.data_as(C.c_void_p), C.c_int32(w.size), bg, _ptr(out.get("trans")),
            _ptr(out.get("final")), _ptr(out.get("depth1")), _ptr(out.get("features10")), _stream(stream)))
        return out

    # ---- S1-S5 (+S7, +S9) ---------------------------------------------------------------
    def make_resolve_desc(self, fb, background, out_trans=None, out_final=None, out_depth1=None,
                          half=None, quarter=None, cell_level=None, level_to_lod=(2, 1, 0, 0),
                          pixel_list=None, pixel_count=None, pass_scales=None,
                          background_image=None):
        """Marshal once, launch many times (the returned object keeps its tensors alive)."""
        d = ResolveDescC()
        d.full = fb.c_struct()
        d.pass_scales = _ptr(pass_scales)
        d.background_image = _ptr(background_image)
        keep = [fb, half, quarter, cell_level, pixel_list, pixel_count, pass_scales, background_image,
                out_trans, out_final,
                out_depth1]
        if half is not None:
            hc = half.c_struct()
            d.half = C.pointer(hc)
            keep.append(hc)
        if quarter is not None:
            qc = quarter.c_struct()
            d.quarter = C.pointer(qc)
            keep.append(qc)
        d.cell_level = _ptr(cell_level)
        d.level_to_lod = (C.c_uint8 * 4)(*level_to_lod)
        d.background = (C.c_float * 3)(*background)
        d.pixel_list, d.pixel_count = _ptr(pixel_list), _ptr(pixel_count)
        d.out_trans, d.out_final, d.out_depth1 = _ptr(out_trans), _ptr(out_final), _ptr(out_depth1)
        d._keep = keep
        return d

    def resolve_desc(self, desc, stream=None):
        self._check(self._L.noit_resolve(self._ctx, C.byref(desc), _stream(stream)))

    def resolve(self, fb: DeviceFragBuf, background=(0.0, 0.0, 0.0), want=("trans", "final", "depth1"),
                out=None, stream=None, **kw):
        """Fused resolve.  Returns dict(trans [P,4], final [P,4], depth1 [P]) of the wanted
        outputs; `out` supplies existing tensors (S9 writes only the listed pixels)."""
        P, dev = fb.num_pixels, fb.offsets.device
        out = dict(out) if out else {}
        for k in want:
            if k not in out:
                out[k] = torch.empty((P,) if k == "depth1" else (P, 4), dtype=torch.float32, device=dev)
        d = self.make_resolve_desc(fb, background, out.get("trans"), out.get("final"),
                                   out.get("depth1"), **kw)
        self.resolve_desc(d, stream)
        return out

    def resolve_host(self, fb_host, background, out_trans=None, out_final=None, out_depth1=None,
                     stream=None):
        """noit_resolve_host: numpy / pinned-tensor HOST buffers in, host buffers out."""
        def hp(a):
            if a is None:
                return None
            return C.c_void_p(a.data_ptr() if isinstance(a, torch.Tensor) else a.ctypes.data)
        d = ResolveDescC()
        d.full = FragBufC(fb_host.width, fb_host.height, int(fb_host.num_fragments),
                          fb_host.color_fmt, hp(fb_host.offsets), hp(fb_host.depth), hp(fb_host.rgba))
        d.level_to_lod = (C.c_uint8 * 4)(2, 1, 0, 0)
        d.background = (C.c_float * 3)(*background)
        d.out_trans, d.out_final, d.out_depth1 = hp(out_trans), hp(out_final), hp(out_depth1)
        self._check(self._L.noit_resolve_host(self._ctx, C.byref(d), _stream(stream)))

    # ---- S6 ---------------------------------------------------------------------------
    def quadtree(self, image: torch.Tensor, width: int, height: int, metric: int = QT_VARIANCE,
                 var_threshold_q: int = 6, corner_threshold: float = 0.02, out=None, stream=None):
        assert image.dtype == torch.float32 and image.is_contiguous()
        dev = image.device
        Tx, Ty = (width + 63) // 64, (height + 63) // 64
        cx, cy = (width + 7) // 8, (height + 7) // 8
        if out is None:
            out = dict(tile_mask=torch.empty(Tx * Ty, dtype=torch.int32, device=dev),
                       cell_level=torch.empty(cx * cy, dtype=torch.uint8, device=dev),
                       hist=torch.empty(4, dtype=torch.int32, device=dev))
        prm = QtParamsC(metric, var_threshold_q, corner_threshold)
        self._check(self._L.noit_quadtree(self._ctx, _ptr(image), C.c_int32(width), C.c_int32(height),
                                          C.byref(prm), _ptr(out["tile_mask"]), _ptr(out["cell_level"]),
                                          _ptr(out["hist"]), _stream(stream)))
        return out

    # ---- NEXT-3 -----------------------------------------------------------------------
    def quadtree16(self, image: torch.Tensor, width: int, height: int, metric: int = QT_CORNER,
                   var_threshold_q: int = 6, corner_threshold: float = 0.02, out=None, stream=None):
        """The paper's tile geometry: 16x16 base tiles down to 2x2 leaves."""
        assert image.dtype == torch.float32 and image.is_contiguous()
        dev = image.device
        Tx, Ty = (width + 15) // 16, (height + 15) // 16
        cx, cy = (width + 1) // 2, (height + 1) // 2
        if out is None:
            out = dict(tile_mask=torch.empty(Tx * Ty, dtype=torch.int32, device=dev),
                       cell_level=torch.empty(cx * cy, dtype=torch.uint8, device=dev),
                       hist=torch.empty(4, dtype=torch.int32, device=dev))
        prm = QtParamsC(metric, var_threshold_q, corner_threshold)
        self._check(self._L.noit_quadtree16(self._ctx, _ptr(image), C.c_int32(width), C.c_int32(height),
                                            C.byref(prm), _ptr(out["tile_mask"]), _ptr(out["cell_level"]),
                                            _ptr(out["hist"]), _stream(stream)))
        return out

    # ---- NEXT-2 -----------------------------------------------------------------------
    def quadtree_temporal(self, image: torch.Tensor, width: int, height: int, prev_mask=None,
                          metric: int = QT_VARIANCE, var_split: int = 6, var_merge: int = 3,
                          corner_split: float = 0.02, corner_merge: float = 0.01, max_step: int = 1,
                          out=None, stream=None):
        assert image.dtype == torch.float32 and image.is_contiguous()
        dev = image.device
        Tx, Ty = (width + 63) // 64, (height + 63) // 64
        cx, cy = (width + 7) // 8, (height + 7) // 8
        if out is None:
            out = dict(tile_mask=torch.empty(Tx * Ty, dtype=torch.int32, device=dev),
                       cell_level=torch.empty(cx * cy, dtype=torch.uint8, device=dev),
                       hist=torch.empty(4, dtype=torch.int32, device=dev))
        prm = QtTemporalParamsC(metric, var_split, var_merge, corner_split, corner_merge, max_step)
        self._check(self._L.noit_quadtree_temporal(
            self._ctx, _ptr(image), C.c_int32(width), C.c_int32(height), C.byref(prm), _ptr(prev_mask),
            _ptr(out["tile_mask"]), _ptr(out["cell_level"]), _ptr(out["hist"]), _stream(stream)))
        return out

    # ---- NEXT-1 -----------------------------------------------------------------------
    def quadtree_balance(self, tile_mask: torch.Tensor, width: int, height: int, iterations: int = 2,
                         delta2: float = 2.2, delta3: float = 3.0, out=None, stream=None,
                         static_scratch: bool = False):
        """In place on `tile_mask`; returns dict(tile_mask, tile_level, cell_level, hist, scales).
        static_scratch=True calls noit_quadtree_balance_static (no allocation inside the call; pass
        `out` so that the binding allocates nothing either; at most 16384 base tiles)."""
        dev = tile_mask.device
        Tx, Ty = (width + 63) // 64, (height + 63) // 64
        cx, cy = (width + 7) // 8, (height + 7) // 8
        if out is None:
            out = dict(tile_level=torch.empty(Tx * Ty, dtype=torch.uint8, device=dev),
                       cell_level=torch.empty(cx * cy, dtype=torch.uint8, device=dev),
                       hist=torch.empty(4, dtype=torch.int32, device=dev),
                       scales=torch.empty(3, dtype=torch.float32, device=dev))
        out["tile_mask"] = tile_mask
        fn = self._L.noit_quadtree_balance_static if static_scratch else self._L.noit_quadtree_balance
        self._check(fn(
            self._ctx, C.c_int32(width), C.c_int32(height), C.c_int32(iterations), C.c_float(delta2),
            C.c_float(delta3), _ptr(tile_mask), _ptr(out["tile_level"]), _ptr(out["cell_level"]),
            _ptr(out["hist"]), _ptr(out["scales"]), _stream(stream)))
        return out

    # ---- S8 ---------------------------------------------------------------------------
    def reproject(self, width, height, M, depth_threshold, background, prev_trans, prev_depth,
                  cur_depth, out=None, stream=None, filter="nearest"):
        import numpy as np
        P, dev = width * height, prev_trans.device
        out = dict(out) if out else {}
        mk = dict(trans=lambda: torch.zeros((P, 4), dtype=torch.float32, device=dev),
                  depth=lambda: torch.zeros(P, dtype=torch.float32, device=dev),
                  final=lambda: torch.zeros((P, 4), dtype=torch.float32, device=dev),
                  accept=lambda: torch.empty(P, dtype=torch.uint8, device=dev),
                  reject_list=lambda: torch.empty(P, dtype=torch.int32, device=dev),
                  reject_count=lambda: torch.empty(1, dtype=torch.int32, device=dev))
        for k, f in mk.items():          # allocate (and zero-fill) only what the caller did not pass
            if k not in out:
                out[k] = f()
        d = ReprojectDescC()
        d.width, d.height = width, height
        d.M = (C.c_float * 16)(*np.asarray(M, np.float32).reshape(-1).tolist())
        d.depth_threshold = depth_threshold
        d.background = (C.c_float * 3)(*background)
        d.prev_trans, d.prev_depth, d.cur_depth = _ptr(prev_trans), _ptr(prev_depth), _ptr(cur_depth)
        d.out_trans, d.out_depth, d.out_final = _ptr(out["trans"]), _ptr(out["depth"]), _ptr(out["final"])
        d.accept, d.reject_list, d.reject_count = (_ptr(out["accept"]), _ptr(out["reject_list"]),
                                                   _ptr(out["reject_count"]))
        d.filter = {"nearest": 0, "bilinear": 1}[filter] if isinstance(filter, str) else int(filter)
        self._check(self._L.noit_reproject(self._ctx, C.byref(d), _stream(stream)))
        return out
