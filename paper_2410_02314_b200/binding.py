"""ctypes binding of libsmlm_b200 (include/smlm.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device
and pinned-host memory and for streams, nothing else.  There is no CPU fallback: if the
shared library is missing it is built (nvcc), and if that fails importing raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

MAX_LAYERS = 32
FP32, BF16, FP16 = 0, 1, 2
TILE_MERGE_NONE, TILE_MERGE_ROW = 0, 1
CONV_AUTO, CONV_TCGEN05, CONV_DIRECT = 0, 1, 2
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED_DEVICE, ERR_CUDA, ERR_OOM, ERR_OVERFLOW = 0, -1, -2, -3, -4, -5
ABI_VERSION = 4
FUSE_AUTO, FUSE_NONE, FUSE_ALL, FUSE_HEAD, FUSE_PAIRS_1CTA = 0, 1, 2, 3, 4
STEM_AUTO, STEM_TENSOR, STEM_CUDA_CORES = 0, 1, 2
KERNEL_STEM, KERNEL_CONV, KERNEL_POST, KERNEL_CONV_PAIR = 0, 1, 2, 3

EXPORTS = ["smlm_create", "smlm_localize", "smlm_check", "smlm_destroy", "smlm_last_error",
           "smlm_launch_count", "smlm_kernel_timing", "smlm_kernel_time_ms",
           "smlm_debug_forward_maps", "smlm_debug_postprocess", "smlm_debug_fill",
           "smlm_ring_open", "smlm_localize_ring", "smlm_ring_acquire", "smlm_ring_release",
           "smlm_ring_close", "smlm_ring_rewind", "smlm_postprocess_static", "smlm_postprocess_static_error"]
RING_PAGEABLE = 1
POST_STATIC_SCRATCH_BYTES = 1048576
POST_STATIC_MAX_TILES = 262080


class NetDesc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("version", C.c_uint32), ("channels", C.c_int32),
                ("n_layers", C.c_int32), ("dilations", C.c_int32 * MAX_LAYERS),
                ("head_channels", C.c_int32), ("precision", C.c_int32), ("stem_relu", C.c_int32),
                ("norm_scale", C.c_float), ("xy_scale", C.c_float), ("z_scale_nm", C.c_float),
                ("photon_scale", C.c_float), ("bg_scale", C.c_float), ("tile", C.c_int32),
                ("micro_batch", C.c_int32), ("conv_impl", C.c_int32),
                ("writeback_frames", C.c_int32), ("fusion", C.c_int32), ("in_frames", C.c_int32),
                ("tile_merge", C.c_int32), ("stem_impl", C.c_int32)]


class PostParams(C.Structure):
    _fields_ = [("head_channels", C.c_int32), ("xy_scale", C.c_float), ("z_scale_nm", C.c_float),
                ("photon_scale", C.c_float), ("bg_scale", C.c_float), ("pixel_size_nm", C.c_float)]


class CameraParams(C.Structure):
    _fields_ = [("pixel_size_nm", C.c_float), ("offset", C.c_float), ("gain", C.c_float),
                ("offset_map", C.c_void_p), ("gain_map", C.c_void_p)]


EMITTER_DTYPE = np.dtype([("frame", "<i4"), ("pix", "<i4"), ("x_nm", "<f4"), ("y_nm", "<f4"),
                          ("z_nm", "<f4"), ("photons", "<f4"), ("bg", "<f4"), ("p", "<f4")])
assert EMITTER_DTYPE.itemsize == 32


class SmlmError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"smlm status {status}: {msg}")
        self.status = status


_LIB = None


def lib():
    """Load (building first if needed) the C-ABI library.  Raises if it cannot be had."""
    global _LIB
    if _LIB is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, i32, i64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_float
        L.smlm_create.restype = C.c_int
        L.smlm_create.argtypes = [C.POINTER(NetDesc), vp, C.POINTER(vp)]
        L.smlm_localize.restype = C.c_int
        L.smlm_localize.argtypes = [vp, vp, i64, i32, i32, C.POINTER(CameraParams), f32, vp,
                                    C.POINTER(i64), vp]
        L.smlm_check.restype = C.c_int
        L.smlm_check.argtypes = [vp]
        L.smlm_destroy.restype = None
        L.smlm_destroy.argtypes = [vp]
        L.smlm_last_error.restype = C.c_char_p
        L.smlm_last_error.argtypes = [vp]
        L.smlm_launch_count.restype = i64
        L.smlm_launch_count.argtypes = [vp]
        L.smlm_kernel_timing.restype = C.c_int
        L.smlm_kernel_timing.argtypes = [vp, i32]
        L.smlm_kernel_time_ms.restype = C.c_int
        L.smlm_kernel_time_ms.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(i64)]
        L.smlm_debug_forward_maps.restype = C.c_int
        L.smlm_debug_forward_maps.argtypes = [vp, vp, i64, i32, i32, C.POINTER(CameraParams), vp,
                                              vp, vp]
        L.smlm_debug_postprocess.restype = C.c_int
        L.smlm_debug_postprocess.argtypes = [vp, vp, i64, i32, i32, C.POINTER(CameraParams), f32,
                                             vp, C.POINTER(i64), vp]
        L.smlm_ring_open.restype = C.c_int
        L.smlm_ring_open.argtypes = [C.c_char_p, i64, i64, i32, i32, i32, i32, i32, i32, C.POINTER(vp)]
        L.smlm_localize_ring.restype = C.c_int
        L.smlm_localize_ring.argtypes = [vp, vp, C.POINTER(CameraParams), f32, vp, C.POINTER(i64), vp]
        L.smlm_ring_acquire.restype = C.c_int
        L.smlm_ring_acquire.argtypes = [vp, C.POINTER(vp), C.POINTER(i64), C.POINTER(i64)]
        L.smlm_ring_release.restype = C.c_int
        L.smlm_ring_release.argtypes = [vp, i64]
        L.smlm_ring_rewind.restype = C.c_int
        L.smlm_ring_rewind.argtypes = [vp]
        L.smlm_ring_close.restype = None
        L.smlm_ring_close.argtypes = [vp]
        L.smlm_debug_fill.restype = C.c_int
        L.smlm_debug_fill.argtypes = [vp, i64, i32, vp]
        L.smlm_postprocess_static.restype = C.c_int
        L.smlm_postprocess_static.argtypes = [vp, i64, i32, i32, C.POINTER(PostParams), f32, vp, i64, vp, vp]
        L.smlm_postprocess_static_error.restype = C.c_char_p
        L.smlm_postprocess_static_error.argtypes = []
        _LIB = L
    return _LIB


def make_desc(channels: int, dilations: Sequence[int], head_channels: int, precision: int,
              stem_relu: int = 1, norm_scale: float = 1000.0, xy_scale: float = 0.5,
              z_scale_nm: float = 700.0, photon_scale: float = 1000.0, bg_scale: float = 100.0,
              tile: int = 0, micro_batch: int = 0, conv_impl: int = CONV_AUTO,
              writeback_frames: int = 0, fusion: int = FUSE_AUTO, in_frames: int = 1,
              tile_merge: int = TILE_MERGE_NONE, stem_impl: int = 0) -> NetDesc:
    d = NetDesc()
    d.struct_size = C.sizeof(NetDesc)
    d.version = ABI_VERSION
    d.channels = int(channels)
    d.n_layers = len(dilations)
    for i, v in enumerate(dilations[:MAX_LAYERS]):
        d.dilations[i] = int(v)
    d.head_channels = int(head_channels)
    d.precision = int(precision)
    d.stem_relu = int(stem_relu)
    d.norm_scale, d.xy_scale, d.z_scale_nm = float(norm_scale), float(xy_scale), float(z_scale_nm)
    d.photon_scale, d.bg_scale = float(photon_scale), float(bg_scale)
    d.tile, d.micro_batch, d.conv_impl = int(tile), int(micro_batch), int(conv_impl)
    d.writeback_frames = int(writeback_frames)
    d.fusion = int(fusion)
    d.in_frames = int(in_frames)
    d.tile_merge = int(tile_merge)
    d.stem_impl = int(stem_impl)
    return d


def desc_from_spec(spec, **overrides) -> NetDesc:
    """spec: smlm_synth.NetSpec (plain data)."""
    kw = dict(channels=spec.channels, dilations=spec.dilations, head_channels=spec.head_channels,
              precision={"bf16": BF16, "fp16": FP16}.get(spec.precision, FP32), stem_relu=spec.stem_relu,
              in_frames=getattr(spec, "in_frames", 1),
              norm_scale=spec.norm_scale, xy_scale=spec.xy_scale, z_scale_nm=spec.z_scale_nm,
              photon_scale=spec.photon_scale, bg_scale=spec.bg_scale)
    kw.update(overrides)
    return make_desc(**kw)


def _ptr(t) -> Optional[int]:
    """Address of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream_handle(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class Localizer:
    """smlm_create / smlm_localize / smlm_destroy with torch tensors as buffers."""

    def __init__(self, desc: NetDesc, weights: np.ndarray):
        self._h = C.c_void_p()
        self.desc = desc
        # out_count words of calls that may still be in flight: the library writes them from a
        # stream-ordered host callback after the call returned, so they must outlive a caller
        # that drops the returned object.  Released by check() / close(), which follow a sync.
        self._counts_in_flight = []
        w = np.ascontiguousarray(weights, dtype="<f4")
        Cc, L, nh = desc.channels, desc.n_layers, desc.head_channels
        IF = 3 if desc.in_frames == 3 else 1
        need = (Cc * IF * 9 + Cc) + L * (Cc * Cc * 9 + Cc) + (nh * Cc + nh)
        if w.size != need:
            raise ValueError(f"weight blob has {w.size} floats, the net needs {need}")
        st = lib().smlm_create(C.byref(desc), w.ctypes.data, C.byref(self._h))
        if st != OK:
            raise SmlmError(st, (lib().smlm_last_error(None) or b"").decode())

    # -- helpers
    def _check(self, st: int):
        if st != OK:
            raise SmlmError(st, self.last_error())

    def last_error(self) -> str:
        return (lib().smlm_last_error(self._h) or b"").decode()

    def camera(self, pixel_size_nm=100.0, offset=100.0, gain=1.0, offset_map=None, gain_map=None):
        cam = CameraParams()
        cam.pixel_size_nm, cam.offset, cam.gain = float(pixel_size_nm), float(offset), float(gain)
        cam.offset_map = _ptr(offset_map)
        cam.gain_map = _ptr(gain_map)
        cam._keep = (offset_map, gain_map)
        return cam

    # -- the hot path
    def localize(self, frames, cam: CameraParams, threshold: float, out_emitters, capacity: int,
                 stream=None, count: Optional[C.c_int64] = None) -> C.c_int64:
        """Enqueue smlm_localize.  frames: uint16 [n][H][W] torch tensor (cuda, or pinned cpu).
        out_emitters: torch uint8/any tensor (cuda or pinned cpu) with >= capacity*32 bytes.
        Returns the ctypes int64 that holds the count once the stream is synchronised."""
        n, H, W = (int(v) for v in frames.shape)
        if count is None:
            count = C.c_int64()
        count.value = int(capacity)
        self._counts_in_flight.append(count)
        st = lib().smlm_localize(self._h, _ptr(frames), n, H, W, C.byref(cam), float(threshold),
                                 _ptr(out_emitters), C.byref(count), _stream_handle(stream))
        self._check(st)
        return count

    def localize_ring(self, ring: "Ring", cam: CameraParams, threshold: float, out_emitters,
                      capacity: int, stream=None, count: Optional[C.c_int64] = None) -> C.c_int64:
        """smlm_localize_ring: the whole frame file behind `ring`, chunk by chunk."""
        if count is None:
            count = C.c_int64()
        count.value = int(capacity)
        self._counts_in_flight.append(count)
        st = lib().smlm_localize_ring(self._h, ring._h, C.byref(cam), float(threshold),
                                      _ptr(out_emitters), C.byref(count), _stream_handle(stream))
        self._check(st)
        return count

    def check(self) -> int:
        """smlm_check; call it after the stream of the last localize has been synchronised."""
        st = lib().smlm_check(self._h)
        self._counts_in_flight.clear()
        return st

    def launch_count(self) -> int:
        return int(lib().smlm_launch_count(self._h))

    def kernel_timing(self, enable: bool):
        self._check(lib().smlm_kernel_timing(self._h, 1 if enable else 0))

    def kernel_time_ms(self, kind: int):
        """(total ms, launches) of KERNEL_STEM / KERNEL_CONV / KERNEL_CONV_PAIR / KERNEL_POST since timing was enabled."""
        ms, k = C.c_double(), C.c_int64()
        self._check(lib().smlm_kernel_time_ms(self._h, int(kind), C.byref(ms), C.byref(k)))
        return ms.value, k.value

    # -- debug exports
    def forward_maps(self, frames, cam: CameraParams, maps, trunk=None, stream=None):
        n, H, W = (int(v) for v in frames.shape)
        st = lib().smlm_debug_forward_maps(self._h, _ptr(frames), n, H, W, C.byref(cam), _ptr(maps),
                                           _ptr(trunk), _stream_handle(stream))
        self._check(st)

    def postprocess(self, maps, cam: CameraParams, threshold: float, out_emitters, capacity: int,
                    stream=None) -> C.c_int64:
        n, nh, H, W = (int(v) for v in maps.shape)
        count = C.c_int64(int(capacity))
        self._counts_in_flight.append(count)
        st = lib().smlm_debug_postprocess(self._h, _ptr(maps), n, H, W, C.byref(cam),
                                          float(threshold), _ptr(out_emitters), C.byref(count),
                                          _stream_handle(stream))
        self._check(st)
        return count

    def close(self):
        if self._h:
            lib().smlm_destroy(self._h)          # synchronises: no callback is pending afterwards
            self._h = C.c_void_p()
            self._counts_in_flight.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


class Ring:
    """smlm_ring_open / smlm_ring_close: reader threads + pinned host ring over a raw uint16
    frame file [n_frames][H][W] (the paper's preloading)."""

    def __init__(self, path: str, n_frames: int, H: int, W: int, chunk_frames: int, n_slots: int = 3,
                 n_threads: int = 2, byte_offset: int = 0, pageable: bool = False):
        self._h = C.c_void_p()
        self.n_frames, self.H, self.W, self.chunk_frames = int(n_frames), int(H), int(W), int(chunk_frames)
        st = lib().smlm_ring_open(os.fsencode(path), int(byte_offset), int(n_frames), int(H), int(W),
                                  int(chunk_frames), int(n_slots), int(n_threads),
                                  RING_PAGEABLE if pageable else 0, C.byref(self._h))
        if st != OK:
            raise SmlmError(st, f"smlm_ring_open({path!r})")

    def acquire(self):
        """-> (numpy view [n][H][W] of the next chunk, first_frame) or (None, None) at the end."""
        p, n, first = C.c_void_p(), C.c_int64(), C.c_int64()
        st = lib().smlm_ring_acquire(self._h, C.byref(p), C.byref(n), C.byref(first))
        if st != OK:
            raise SmlmError(st, "smlm_ring_acquire")
        if n.value == 0:
            return None, None
        arr = np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_uint16)), shape=(n.value, self.H, self.W))
        return arr, first.value

    def release(self, first_frame: int):
        st = lib().smlm_ring_release(self._h, int(first_frame))
        if st != OK:
            raise SmlmError(st, "smlm_ring_release")

    def rewind(self):
        """Start over at the first chunk (every acquired chunk must have been released)."""
        st = lib().smlm_ring_rewind(self._h)
        if st != OK:
            raise SmlmError(st, "smlm_ring_rewind")

    def close(self):
        if self._h:
            lib().smlm_ring_close(self._h)
            self._h = C.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def postprocess_static(maps, head_channels: int, threshold: float, out_emitters, capacity: int, out_count,
                       xy_scale: float = 0.5, z_scale_nm: float = 700.0, photon_scale: float = 1000.0,
                       bg_scale: float = 100.0, pixel_size_nm: float = 100.0, stream=None,
                       shape: Optional[Sequence[int]] = None) -> None:
    """smlm_postprocess_static: post-processing without a ctx and without any GPU allocation
    (for callers that cannot call cudaMalloc: see include/smlm.h).  maps: cuda float32
    [n][head_channels][H][W] (or a raw address plus `shape` = (n, H, W)); out_emitters: cuda
    buffer of capacity * 32 bytes; out_count: cuda int64 tensor of one element, written by the
    GPU.  Enqueues only; raises SmlmError with the library's message on a refused call."""
    if shape is None:
        n, nh, H, W = (int(v) for v in maps.shape)
        if nh != head_channels:
            raise ValueError("maps.shape[1] != head_channels")
    else:
        n, H, W = (int(v) for v in shape)
    pp = PostParams(int(head_channels), float(xy_scale), float(z_scale_nm), float(photon_scale),
                    float(bg_scale), float(pixel_size_nm))
    st = lib().smlm_postprocess_static(_ptr(maps), n, H, W, C.byref(pp), float(threshold), _ptr(out_emitters),
                                       int(capacity), _ptr(out_count), _stream_handle(stream))
    if st != OK:
        raise SmlmError(st, (lib().smlm_postprocess_static_error() or b"").decode())


def debug_fill(buf, mode: int, stream=None) -> None:
    """smlm_debug_fill over a whole cuda tensor (mode 0: cudaMemsetAsync, 1: 16-byte store kernel)."""
    st = lib().smlm_debug_fill(_ptr(buf), int(buf.numel() * buf.element_size()), int(mode), _stream_handle(stream))
    if st != OK:
        raise SmlmError(st, "smlm_debug_fill")


def emitters_to_numpy(buf, count: int) -> np.ndarray:
    """View the first `count` records of a torch byte/any tensor as a structured array (copy),
    sorted by (frame, pix) - the canonical order for comparison (order is unspecified)."""
    t = buf.detach().cpu().contiguous().view(-1)
    raw = t.numpy().view(np.uint8)[: int(count) * 32].copy()
    em = raw.view(EMITTER_DTYPE)
    return em[np.lexsort((em["pix"], em["frame"]))]
