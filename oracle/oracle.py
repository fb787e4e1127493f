"""ctypes wrapper around oracle/smlm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` leg
may import this module.  It imports nothing from paper_2410_02314_b200/.

The C file is compiled on the machine that runs it (gcc -O3 -march=native -fopenmp) into
oracle/_build/, keyed by the host's CPU flags, because the box that builds the repo and
the box that runs the GPU tests need not have the same CPU.
"""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "smlm_oracle.c")
_BUILD = os.path.join(_HERE, "_build")
MAX_LAYERS = 32


class OracleNet(C.Structure):
    _fields_ = [("channels", C.c_int32), ("n_layers", C.c_int32),
                ("dilations", C.c_int32 * MAX_LAYERS), ("head_channels", C.c_int32),
                ("stem_relu", C.c_int32), ("norm_scale", C.c_double), ("xy_scale", C.c_double),
                ("z_scale_nm", C.c_double), ("photon_scale", C.c_double), ("bg_scale", C.c_double),
                ("in_frames", C.c_int32)]


class OracleCamera(C.Structure):
    _fields_ = [("pixel_size_nm", C.c_double), ("offset", C.c_double), ("gain", C.c_double),
                ("offset_map", C.POINTER(C.c_float)), ("gain_map", C.POINTER(C.c_float))]


class OracleEmitter(C.Structure):
    _fields_ = [("frame", C.c_int32), ("pix", C.c_int32), ("x_nm", C.c_double),
                ("y_nm", C.c_double), ("z_nm", C.c_double), ("photons", C.c_double),
                ("bg", C.c_double), ("p", C.c_double)]


EMITTER_DTYPE = np.dtype([("frame", "<i4"), ("pix", "<i4"), ("x_nm", "<f8"), ("y_nm", "<f8"),
                          ("z_nm", "<f8"), ("photons", "<f8"), ("bg", "<f8"), ("p", "<f8")])
assert EMITTER_DTYPE.itemsize == C.sizeof(OracleEmitter)


def _cpu_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo", "r", encoding="utf-8") as fh:
            for line in fh:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    with open(_SRC, "rb") as fh:
        src = fh.read()
    return hashlib.sha1(flags.encode() + src).hexdigest()[:12]


def build(verbose: bool = False) -> str:
    """Compile smlm_oracle.c for this host if not already done; return the .so path."""
    os.makedirs(_BUILD, exist_ok=True)
    so = os.path.join(_BUILD, f"libsmlm_oracle_{_cpu_tag()}.so")
    if not os.path.exists(so):
        tmp = so + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=c11",
               "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        if verbose:
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
        os.replace(tmp, so)
    return so


_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(build())
        L.smlm_oracle_threads.restype = C.c_int
        L.smlm_oracle_blob_size.restype = C.c_int64
        L.smlm_oracle_blob_size.argtypes = [C.POINTER(OracleNet)]
        L.smlm_oracle_forward_maps.restype = C.c_int
        L.smlm_oracle_forward_maps.argtypes = [C.POINTER(OracleNet), C.c_void_p, C.c_void_p,
                                               C.c_int64, C.c_int, C.c_int,
                                               C.POINTER(OracleCamera), C.c_void_p, C.c_void_p]
        L.smlm_oracle_activate_maps.restype = C.c_int
        L.smlm_oracle_activate_maps.argtypes = [C.POINTER(OracleNet), C.c_void_p, C.c_int64,
                                                C.c_int, C.c_int, C.c_void_p]
        L.smlm_oracle_postprocess.restype = C.c_int
        L.smlm_oracle_postprocess.argtypes = [C.POINTER(OracleNet), C.c_void_p, C.c_int64, C.c_int,
                                              C.c_int, C.POINTER(OracleCamera), C.c_double,
                                              C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
        _LIB = L
    return _LIB


def threads() -> int:
    return int(lib().smlm_oracle_threads())


def make_net(channels: int, dilations: Sequence[int], head_channels: int, stem_relu: int = 1,
             norm_scale: float = 1000.0, xy_scale: float = 0.5, z_scale_nm: float = 700.0,
             photon_scale: float = 1000.0, bg_scale: float = 100.0, in_frames: int = 1) -> OracleNet:
    net = OracleNet()
    net.channels = int(channels)
    net.n_layers = len(dilations)
    for i, d in enumerate(dilations):
        net.dilations[i] = int(d)
    net.head_channels = int(head_channels)
    net.stem_relu = int(stem_relu)
    net.norm_scale = float(norm_scale)
    net.xy_scale = float(xy_scale)
    net.z_scale_nm = float(z_scale_nm)
    net.photon_scale = float(photon_scale)
    net.bg_scale = float(bg_scale)
    net.in_frames = int(in_frames)
    return net


def net_from_spec(spec) -> OracleNet:
    """spec: smlm_synth.NetSpec (plain data)."""
    return make_net(spec.channels, spec.dilations, spec.head_channels, spec.stem_relu,
                    spec.norm_scale, spec.xy_scale, spec.z_scale_nm, spec.photon_scale,
                    spec.bg_scale, getattr(spec, "in_frames", 1))


class _Cam:
    """Keeps the float32 maps alive next to the ctypes struct."""

    def __init__(self, pixel_size_nm, offset, gain, offset_map, gain_map):
        self.off = None if offset_map is None else np.ascontiguousarray(offset_map, dtype=np.float32)
        self.gain = None if gain_map is None else np.ascontiguousarray(gain_map, dtype=np.float32)
        self.c = OracleCamera()
        self.c.pixel_size_nm = float(pixel_size_nm)
        self.c.offset = float(offset)
        self.c.gain = float(gain)
        fp = C.POINTER(C.c_float)
        self.c.offset_map = self.off.ctypes.data_as(fp) if self.off is not None else fp()
        self.c.gain_map = self.gain.ctypes.data_as(fp) if self.gain is not None else fp()


def make_camera(pixel_size_nm=100.0, offset=100.0, gain=1.0, offset_map=None, gain_map=None) -> _Cam:
    return _Cam(pixel_size_nm, offset, gain, offset_map, gain_map)


def forward_maps(net: OracleNet, weights: np.ndarray, frames: np.ndarray, cam: _Cam,
                 dump_trunk: bool = False):
    """O1-O4.  Returns o [n][n_h][H][W] float64 (pre-activation); with dump_trunk also
    a [n][L+1][H][W][C]."""
    frames = np.ascontiguousarray(frames, dtype=np.uint16)
    assert frames.ndim == 3
    n, H, W = frames.shape
    w = np.ascontiguousarray(weights, dtype=np.float32)
    assert w.size == lib().smlm_oracle_blob_size(C.byref(net)), "weight blob size mismatch"
    if cam.off is not None:
        assert cam.off.shape == (H, W) and cam.gain.shape == (H, W)
    out = np.empty((n, net.head_channels, H, W), dtype=np.float64)
    dump = np.empty((n, net.n_layers + 1, H, W, net.channels), dtype=np.float64) if dump_trunk else None
    rc = lib().smlm_oracle_forward_maps(C.byref(net), w.ctypes.data, frames.ctypes.data, n, H, W,
                                        C.byref(cam.c), out.ctypes.data,
                                        dump.ctypes.data if dump is not None else None)
    if rc != 0:
        raise RuntimeError(f"smlm_oracle_forward_maps failed ({rc})")
    return (out, dump) if dump_trunk else out


def activate_maps(net: OracleNet, o: np.ndarray) -> np.ndarray:
    """O5 on whole maps: p, xy_scale*tanh, tanh (z), softplus (N, bg)."""
    o = np.ascontiguousarray(o, dtype=np.float64)
    n, nh, H, W = o.shape
    assert nh == net.head_channels
    act = np.empty_like(o)
    rc = lib().smlm_oracle_activate_maps(C.byref(net), o.ctypes.data, n, H, W, act.ctypes.data)
    if rc != 0:
        raise RuntimeError("smlm_oracle_activate_maps failed")
    return act


def postprocess(net: OracleNet, o: np.ndarray, cam: _Cam, threshold: float,
                capacity: Optional[int] = None) -> np.ndarray:
    """O6-O8.  Returns a structured array (EMITTER_DTYPE) sorted by (frame, pix)."""
    o = np.ascontiguousarray(o, dtype=np.float64)
    n, nh, H, W = o.shape
    assert nh == net.head_channels
    if capacity is None:
        capacity = n * ((H + 1) // 2) * ((W + 1) // 2)   # no two detections are 8-adjacent
    buf = np.zeros(max(capacity, 1), dtype=EMITTER_DTYPE)
    cnt = C.c_int64(0)
    rc = lib().smlm_oracle_postprocess(C.byref(net), o.ctypes.data, n, H, W, C.byref(cam.c),
                                       float(threshold), buf.ctypes.data, capacity, C.byref(cnt))
    if rc != 0:
        raise RuntimeError("smlm_oracle_postprocess failed")
    assert cnt.value <= capacity, "oracle capacity bound violated"
    return buf[:cnt.value].copy()


def localize(net: OracleNet, weights: np.ndarray, frames: np.ndarray, cam: _Cam, threshold: float):
    """The whole path O1-O8: frames -> emitter list."""
    return postprocess(net, forward_maps(net, weights, frames, cam), cam, threshold)
