"""ctypes wrapper around oracle/dloc_oracle.c (the paper's own DilatedLoc topology, SURVEY.md
8(f)-2) -- TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/ may import this module; it imports
nothing from paper_2410_02314_b200/.  Detection and decode of the first six heads are the
rule of smlm_oracle.c (O6-O8), called through oracle.oracle; the uncertainty heads are decoded
here."""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess
from typing import Sequence

import numpy as np

from . import oracle as O

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dloc_oracle.c")
_BUILD = os.path.join(_HERE, "_build")
HEADS = 10


class DlocNet(C.Structure):
    _fields_ = [("c0", C.c_int32), ("growth", C.c_int32), ("n_blocks", C.c_int32), ("n_dil", C.c_int32),
                ("dilations", C.c_int32 * 8), ("in_frames", C.c_int32), ("stem_relu", C.c_int32),
                ("norm_scale", C.c_double)]


class DlocCamera(C.Structure):
    _fields_ = [("pixel_size_nm", C.c_double), ("offset", C.c_double), ("gain", C.c_double),
                ("offset_map", C.POINTER(C.c_float)), ("gain_map", C.POINTER(C.c_float))]


def build() -> str:
    os.makedirs(_BUILD, exist_ok=True)
    flags = ""
    try:
        with open("/proc/cpuinfo", "r", encoding="utf-8") as fh:
            flags = next((l for l in fh if l.startswith("flags")), "")
    except OSError:
        pass
    with open(_SRC, "rb") as fh:
        tag = hashlib.sha1(flags.encode() + fh.read()).hexdigest()[:12]
    so = os.path.join(_BUILD, f"libdloc_oracle_{tag}.so")
    if not os.path.exists(so):
        tmp = so + f".tmp{os.getpid()}"
        subprocess.run(["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-Wall",
                        "-Wextra", "-o", tmp, _SRC, "-lm"], check=True)
        os.replace(tmp, so)
    return so


_LIB = None


def lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(build())
        L.dloc_oracle_blob_size.restype = C.c_int64
        L.dloc_oracle_blob_size.argtypes = [C.POINTER(DlocNet)]
        L.dloc_oracle_forward_maps.restype = C.c_int
        L.dloc_oracle_forward_maps.argtypes = [C.POINTER(DlocNet), C.c_void_p, C.c_void_p, C.c_int64, C.c_int,
                                               C.c_int, C.POINTER(DlocCamera), C.c_void_p, C.c_void_p]
        L.dloc_oracle_sigmas.restype = C.c_int
        L.dloc_oracle_sigmas.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int64,
                                         C.c_double, C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.dloc_oracle_maxpool2.restype = C.c_int
        L.dloc_oracle_maxpool2.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.dloc_oracle_upsample2.restype = C.c_int
        L.dloc_oracle_upsample2.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        _LIB = L
    return _LIB


def maxpool2(x: np.ndarray) -> np.ndarray:
    """The oracle's 2 x 2 / stride 2 / floor max pooling (reading D4) of a planar [c][H][W] map."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    c, H, W = x.shape
    out = np.empty((c, H // 2, W // 2), np.float64)
    if lib().dloc_oracle_maxpool2(x.ctypes.data, c, H, W, out.ctypes.data) != 0:
        raise ValueError("dloc_oracle_maxpool2: bad argument")
    return out


def upsample2(x: np.ndarray, Ho: int, Wo: int) -> np.ndarray:
    """The oracle's nearest-neighbour x 2 up-sampling to exactly Ho x Wo (reading D5)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    c, H, W = x.shape
    out = np.empty((c, int(Ho), int(Wo)), np.float64)
    if lib().dloc_oracle_upsample2(x.ctypes.data, c, H, W, int(Ho), int(Wo), out.ctypes.data) != 0:
        raise ValueError("dloc_oracle_upsample2: bad argument")
    return out


def make_net(c0: int, growth: int, n_blocks: int = 4, dilations: Sequence[int] = (2, 4, 8, 16),
             in_frames: int = 1, stem_relu: int = 1, norm_scale: float = 1000.0) -> DlocNet:
    net = DlocNet()
    net.c0, net.growth, net.n_blocks, net.n_dil = int(c0), int(growth), int(n_blocks), len(dilations)
    for i, d in enumerate(dilations):
        net.dilations[i] = int(d)
    net.in_frames, net.stem_relu, net.norm_scale = int(in_frames), int(stem_relu), float(norm_scale)
    return net


def net_from_spec(spec) -> DlocNet:
    """spec: smlm_synth.DlocSpec (plain data)."""
    return make_net(spec.c0, spec.growth, spec.n_blocks, spec.dilations, spec.in_frames, spec.stem_relu,
                    spec.norm_scale)


def blob_size(net: DlocNet) -> int:
    return int(lib().dloc_oracle_blob_size(C.byref(net)))


def dump_shapes(net: DlocNet, H: int, W: int):
    """Names and planar shapes of the feature maps in the dump of forward_maps."""
    c = net.c0
    out = [("stem", (c, H, W))] + [(f"block{b}", (c, H, W)) for b in range(net.n_blocks)]
    out += [("e1", (2 * c, H // 2, W // 2)), ("e2", (4 * c, H // 4, W // 4)), ("m1", (2 * c, H // 2, W // 2)),
            ("m0", (c, H, W))]
    return out


def forward_maps(net: DlocNet, weights: np.ndarray, frames: np.ndarray, cam, dump: bool = False):
    """-> o [n][10][H][W] float64 (pre-activation) [, list per frame of {name: planar map}]."""
    frames = np.ascontiguousarray(frames, dtype=np.uint16)
    n, H, W = frames.shape
    w = np.ascontiguousarray(weights, dtype=np.float32)
    assert w.size == blob_size(net), (w.size, blob_size(net))
    c = DlocCamera()
    c.pixel_size_nm, c.offset, c.gain = cam.c.pixel_size_nm, cam.c.offset, cam.c.gain
    c.offset_map, c.gain_map = cam.c.offset_map, cam.c.gain_map
    out = np.empty((n, HEADS, H, W), dtype=np.float64)
    shapes = dump_shapes(net, H, W)
    per = sum(int(np.prod(s)) for _, s in shapes)
    buf = np.empty((n, per), dtype=np.float64) if dump else None
    rc = lib().dloc_oracle_forward_maps(C.byref(net), w.ctypes.data, frames.ctypes.data, n, H, W, C.byref(c),
                                        out.ctypes.data, buf.ctypes.data if dump else None)
    if rc != 0:
        raise RuntimeError("dloc_oracle_forward_maps failed")
    if not dump:
        return out
    maps = []
    for f in range(n):
        d, off = {}, 0
        for name, s in shapes:
            k = int(np.prod(s))
            d[name] = buf[f, off:off + k].reshape(s)
            off += k
        maps.append(d)
    return out, maps


UNC_DTYPE = np.dtype(O.EMITTER_DTYPE.descr + [("sx_nm", "<f8"), ("sy_nm", "<f8"), ("sz_nm", "<f8"),
                                               ("s_photons", "<f8")])


def postprocess(spec, o: np.ndarray, cam, threshold: float) -> np.ndarray:
    """Detection + decode on o [n][10][H][W]: heads 0-5 by the rule of smlm_oracle.c (O6-O8, the
    six-head layout p, dx, dy, z, N, bg), heads 6-9 the uncertainties (reading D7)."""
    o = np.ascontiguousarray(o, dtype=np.float64)
    n, nh, H, W = o.shape
    assert nh == HEADS
    net6 = O.make_net(spec.c0, (1,), 6, 1, spec.norm_scale, spec.xy_scale, spec.z_scale_nm, spec.photon_scale,
                      spec.bg_scale)
    em = O.postprocess(net6, np.ascontiguousarray(o[:, :6]), cam, threshold)
    out = np.zeros(len(em), dtype=UNC_DTYPE)
    for k in O.EMITTER_DTYPE.names:
        out[k] = em[k]
    sig = np.zeros((len(em), 4), dtype=np.float64)
    fr = np.ascontiguousarray(em["frame"], dtype=np.int32)
    px = np.ascontiguousarray(em["pix"], dtype=np.int32)
    rc = lib().dloc_oracle_sigmas(o.ctypes.data, H, W, fr.ctypes.data, px.ctypes.data, len(em),
                                  float(cam.c.pixel_size_nm), float(spec.sigma_xy_px), float(spec.sigma_z_nm),
                                  float(spec.sigma_photons), sig.ctypes.data)
    if rc != 0:
        raise RuntimeError("dloc_oracle_sigmas failed")
    for i, k in enumerate(("sx_nm", "sy_nm", "sz_nm", "s_photons")):
        out[k] = sig[:, i]
    return out
