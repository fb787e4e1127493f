"""ctypes binding of the DilatedLoc entry points of libsmlm_b200 (include/dloc.h): argument
marshalling only.  Every step runs in the library's CUDA kernels; there is no CPU fallback."""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from . import binding as B

DLOC_ABI_VERSION = 1
DLOC_HEADS = 10
DLOC_MAX_DIL = 8
DLOC_EXPORTS = ["dloc_create", "dloc_localize", "dloc_debug_forward_maps", "dloc_check", "dloc_last_error",
                "dloc_launch_count", "dloc_kernel_timing", "dloc_conv_time_ms", "dloc_destroy"]


class DlocDesc(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("version", C.c_uint32), ("c0", C.c_int32), ("growth", C.c_int32),
                ("n_blocks", C.c_int32), ("n_dil", C.c_int32), ("dilations", C.c_int32 * DLOC_MAX_DIL),
                ("in_frames", C.c_int32), ("stem_relu", C.c_int32), ("precision", C.c_int32),
                ("norm_scale", C.c_float), ("xy_scale", C.c_float), ("z_scale_nm", C.c_float),
                ("photon_scale", C.c_float), ("bg_scale", C.c_float), ("sigma_xy_px", C.c_float),
                ("sigma_z_nm", C.c_float), ("sigma_photons", C.c_float), ("micro_batch", C.c_int32),
                ("conv_impl", C.c_int32)]


DLOC_EMITTER_DTYPE = np.dtype(B.EMITTER_DTYPE.descr + [("sx_nm", "<f4"), ("sy_nm", "<f4"), ("sz_nm", "<f4"),
                                                        ("s_photons", "<f4")])
assert DLOC_EMITTER_DTYPE.itemsize == 48

_READY = False


def dlib():
    global _READY
    L = B.lib()
    if not _READY:
        vp, i32, i64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_float
        L.dloc_create.restype = C.c_int
        L.dloc_create.argtypes = [C.POINTER(DlocDesc), vp, C.POINTER(vp)]
        L.dloc_localize.restype = C.c_int
        L.dloc_localize.argtypes = [vp, vp, i64, i32, i32, C.POINTER(B.CameraParams), f32, vp, C.POINTER(i64), vp]
        L.dloc_debug_forward_maps.restype = C.c_int
        L.dloc_debug_forward_maps.argtypes = [vp, vp, i64, i32, i32, C.POINTER(B.CameraParams), vp, vp, vp]
        L.dloc_check.restype = C.c_int
        L.dloc_check.argtypes = [vp]
        L.dloc_last_error.restype = C.c_char_p
        L.dloc_last_error.argtypes = [vp]
        L.dloc_launch_count.restype = i64
        L.dloc_launch_count.argtypes = [vp]
        L.dloc_kernel_timing.restype = C.c_int
        L.dloc_kernel_timing.argtypes = [vp, i32]
        L.dloc_conv_time_ms.restype = C.c_int
        L.dloc_conv_time_ms.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
        L.dloc_destroy.restype = None
        L.dloc_destroy.argtypes = [vp]
        _READY = True
    return L


def dloc_desc(c0: int, growth: int, n_blocks: int = 4, dilations: Sequence[int] = (2, 4, 8, 16), in_frames: int = 1,
              stem_relu: int = 1, precision: int = B.BF16, norm_scale: float = 1000.0, xy_scale: float = 0.5,
              z_scale_nm: float = 700.0, photon_scale: float = 1000.0, bg_scale: float = 100.0,
              sigma_xy_px: float = 3.0, sigma_z_nm: float = 700.0, sigma_photons: float = 1000.0,
              micro_batch: int = 0, conv_impl: int = B.CONV_AUTO) -> DlocDesc:
    d = DlocDesc()
    d.struct_size, d.version = C.sizeof(DlocDesc), DLOC_ABI_VERSION
    d.c0, d.growth, d.n_blocks, d.n_dil = int(c0), int(growth), int(n_blocks), len(dilations)
    for i, v in enumerate(dilations[:DLOC_MAX_DIL]):
        d.dilations[i] = int(v)
    d.in_frames, d.stem_relu, d.precision = int(in_frames), int(stem_relu), int(precision)
    d.norm_scale, d.xy_scale, d.z_scale_nm = float(norm_scale), float(xy_scale), float(z_scale_nm)
    d.photon_scale, d.bg_scale = float(photon_scale), float(bg_scale)
    d.sigma_xy_px, d.sigma_z_nm, d.sigma_photons = float(sigma_xy_px), float(sigma_z_nm), float(sigma_photons)
    d.micro_batch, d.conv_impl = int(micro_batch), int(conv_impl)
    return d


def dloc_desc_from_spec(spec, **overrides) -> DlocDesc:
    """spec: smlm_synth.DlocSpec (plain data)."""
    kw = dict(c0=spec.c0, growth=spec.growth, n_blocks=spec.n_blocks, dilations=spec.dilations,
              in_frames=spec.in_frames, stem_relu=spec.stem_relu,
              precision={"bf16": B.BF16, "fp16": B.FP16}.get(spec.precision, B.FP32), norm_scale=spec.norm_scale,
              xy_scale=spec.xy_scale, z_scale_nm=spec.z_scale_nm, photon_scale=spec.photon_scale,
              bg_scale=spec.bg_scale, sigma_xy_px=spec.sigma_xy_px, sigma_z_nm=spec.sigma_z_nm,
              sigma_photons=spec.sigma_photons)
    kw.update(overrides)
    return dloc_desc(**kw)


class DlocLocalizer:
    """dloc_create / dloc_localize / dloc_destroy with torch tensors as buffers."""

    def __init__(self, desc: DlocDesc, weights: np.ndarray):
        self._h = C.c_void_p()
        self.desc = desc
        w = np.ascontiguousarray(weights, dtype="<f4")
        self._counts_in_flight = []
        st = dlib().dloc_create(C.byref(desc), w.ctypes.data, C.byref(self._h))
        if st != B.OK:
            raise B.SmlmError(st, (dlib().dloc_last_error(None) or b"").decode())

    def _check(self, st: int):
        if st != B.OK:
            raise B.SmlmError(st, self.last_error())

    def last_error(self) -> str:
        return (dlib().dloc_last_error(self._h) or b"").decode()

    def camera(self, pixel_size_nm=100.0, offset=100.0, gain=1.0, offset_map=None, gain_map=None):
        cam = B.CameraParams()
        cam.pixel_size_nm, cam.offset, cam.gain = float(pixel_size_nm), float(offset), float(gain)
        cam.offset_map = B._ptr(offset_map)
        cam.gain_map = B._ptr(gain_map)
        cam._keep = (offset_map, gain_map)
        return cam

    def localize(self, frames, cam, threshold: float, out_emitters, capacity: int, stream=None,
                 count: Optional[C.c_int64] = None) -> C.c_int64:
        n, H, W = (int(v) for v in frames.shape)
        if count is None:
            count = C.c_int64()
        count.value = int(capacity)
        self._counts_in_flight.append(count)     # written by a stream callback after the call returned
        st = dlib().dloc_localize(self._h, B._ptr(frames), n, H, W, C.byref(cam), float(threshold),
                                  B._ptr(out_emitters), C.byref(count), B._stream_handle(stream))
        self._check(st)
        return count

    def forward_maps(self, frames, cam, maps, dump=None, stream=None):
        n, H, W = (int(v) for v in frames.shape)
        self._check(dlib().dloc_debug_forward_maps(self._h, B._ptr(frames), n, H, W, C.byref(cam), B._ptr(maps),
                                                   B._ptr(dump), B._stream_handle(stream)))

    def check(self) -> int:
        """dloc_check; call it after the stream of the last localize has been synchronised."""
        st = dlib().dloc_check(self._h)
        self._counts_in_flight.clear()
        return st

    def launch_count(self) -> int:
        return int(dlib().dloc_launch_count(self._h))

    def kernel_timing(self, enable: bool):
        self._check(dlib().dloc_kernel_timing(self._h, 1 if enable else 0))

    def conv_time_ms(self):
        ms, k = C.c_double(), C.c_int64()
        self._check(dlib().dloc_conv_time_ms(self._h, C.byref(ms), C.byref(k)))
        return ms.value, k.value

    def close(self):
        if self._h:
            dlib().dloc_destroy(self._h)
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


def dloc_emitters_to_numpy(buf, count: int) -> np.ndarray:
    """torch uint8 buffer (cuda or cpu) -> structured array sorted by (frame, pix) (presentation only)."""
    raw = buf.detach().cpu().numpy().view(np.uint8)[: int(count) * 48]
    em = np.frombuffer(raw.tobytes(), dtype=DLOC_EMITTER_DTYPE).copy()
    return em[np.lexsort((em["pix"], em["frame"]))]
