"""Seeded synthetic weights (inputs only; no arithmetic of the method).

Trained DilatedLoc weights are not available, so every config runs
on random-init weights of the named architecture: "Weights are He-normal from the seed
and biases are zero" (BASELINE.json configs[0]).

Blob layout (one little-endian fp32 array, the `weights` argument of smlm_create and of
the oracle; include/smlm.h):
    stem  W[C][1][3][3], b[C]
    for l in 0..L-1:  W_l[C_out][C_in][3][3], b_l[C]
    head  W[n_h][C], b[n_h]
OIHW, cross-correlation (reading G2).  Draw order == blob order (reading G11):
std = sqrt(2 / fan_in), fan_in = C_in * 3 * 3 (stem 9, trunk 9C, head C).

Flavours (readings G12, G13 of SURVEY.md 8(c), restated in DESIGN.md):
  "literal"  He-normal, zero biases, nothing else.  cfg 0.
  "lc"       trunk weights x g_res (= 1/sqrt(L)); head rows x row_gain[h]; p-head row x kappa
             and bias b_p.  kappa, b_p, row_gain come from `calibration.json`, which is
             written by tests/golden/make_calibration.py from ORACLE statistics only
             (never from the CUDA path).  Low-contrast set used in bf16 mode.
  "hc"       same with a high-contrast p-head (logit std 3) - the strong index test, run
             through the library's fp32 mode.
  "st"       surrogate for TRAINED weights ("the probability of a
             fluorescent molecule" peaks at single pixels): hand-set signal channels inside the
             random net, so that the p-map has sharp peaks at the emitters and ~1 % of the
             pixels exceed the threshold, as a trained DilatedLoc would give, instead of the
             smooth map of random weights.  Stem channel 0 is a zero-mean matched filter for the
             sigma = 1.3 px PSF, channels 1-4 are +x / -x / +y / -y gradient filters; the trunk
             rows that write into these five channels are scaled by `ST_TRUNK_LEAK`; the p-head
             reads channel 0 only (x kappa, + b_p from calibration.json, oracle statistics), the
             dx / dy heads read the gradient channels, the other rows are the random ones x 0.3.
             Everything else (the other stem filters, the trunk) is the seeded He-normal draw.
The library never sees flavours: it receives the final blob.
"""
from __future__ import annotations

import json
import os
from typing import Optional

import numpy as np

from .configs import Config, NetSpec

_CALIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "calibration.json")


def blob_size(net: NetSpec) -> int:
    return net.n_params()


def blob_offsets(net: NetSpec) -> dict:
    """Element offsets of every tensor inside the blob."""
    C, L, nh = net.channels, net.n_layers, net.head_channels
    off = {}
    p = 0
    off["stem_w"] = p; p += C * net.in_frames * 9
    off["stem_b"] = p; p += C
    for l in range(L):
        off[f"w{l}"] = p; p += C * C * 9
        off[f"b{l}"] = p; p += C
    off["head_w"] = p; p += nh * C
    off["head_b"] = p; p += nh
    assert p == blob_size(net)
    return off


def he_normal_blob(net: NetSpec, seed: int) -> np.ndarray:
    """The literal reading: He-normal weights in blob order, zero biases."""
    C, L, nh = net.channels, net.n_layers, net.head_channels
    rng = np.random.default_rng([int(seed), 0x57E1])
    parts = []
    parts.append(rng.normal(0.0, np.sqrt(2.0 / (9.0 * net.in_frames)), size=C * net.in_frames * 9))
    parts.append(np.zeros(C))
    for _ in range(L):
        parts.append(rng.normal(0.0, np.sqrt(2.0 / (9.0 * C)), size=C * C * 9))
        parts.append(np.zeros(C))
    parts.append(rng.normal(0.0, np.sqrt(2.0 / C), size=nh * C))
    parts.append(np.zeros(nh))
    return np.concatenate(parts).astype(np.float32)


def load_calibration() -> dict:
    if not os.path.exists(_CALIB_PATH):
        return {}
    with open(_CALIB_PATH, "r", encoding="utf-8") as fh:
        return json.load(fh)


def calibration_key(cfg: Config, flavour: str, seed: int) -> str:
    return f"cfg{cfg.index}/{flavour}/seed{int(seed)}"


def apply_recipe(net: NetSpec, blob: np.ndarray, g_res: float, row_gain, kappa: float,
                 b_p: float) -> np.ndarray:
    """Scale trunk by g_res, head row h by row_gain[h], p-row additionally by kappa; set b_p."""
    out = blob.astype(np.float64).copy()
    off = blob_offsets(net)
    C, L, nh = net.channels, net.n_layers, net.head_channels
    for l in range(L):
        s = off[f"w{l}"]
        out[s:s + C * C * 9] *= g_res
    hw = off["head_w"]
    for h in range(nh):
        g = float(row_gain[h]) * (float(kappa) if h == 0 else 1.0)
        out[hw + h * C: hw + (h + 1) * C] *= g
    out[off["head_b"] + 0] = b_p
    return out.astype(np.float32)


ST_SIGNAL_GAIN = 4.0     # scale of the five hand-set stem filters
ST_TRUNK_LEAK = 0.05     # trunk rows writing into the signal channels: residual additions stay small
ST_XY_GAIN = 2.0         # dx / dy head gain on the gradient channels


def st_base_blob(net: NetSpec, seed: int, g_res: float, sigma_px: float = 1.3) -> np.ndarray:
    """The "st" flavour before calibration (p-head = channel 0 with gain 1 and zero bias)."""
    out = he_normal_blob(net, seed).astype(np.float64)
    off = blob_offsets(net)
    C, L, nh, IF = net.channels, net.n_layers, net.head_channels, net.in_frames
    k = np.arange(-1, 2, dtype=np.float64)
    g = np.exp(-(k[:, None] ** 2 + k[None, :] ** 2) / (2.0 * sigma_px ** 2))
    mf = g - g.mean()
    mf /= np.sqrt((mf ** 2).sum())
    gx = np.outer([1.0, 2.0, 1.0], [-1.0, 0.0, 1.0]) / 8.0          # [ky][kx]: rises to the right
    stem = out[off["stem_w"]:off["stem_w"] + C * IF * 9].reshape(C, IF, 3, 3)
    stem[:5] = 0.0
    c = IF // 2                                                        # the frame itself (3-frame context: centre)
    for ch, f in enumerate((mf, gx, -gx, gx.T, -gx.T)):
        stem[ch, c] = ST_SIGNAL_GAIN * f
    for l in range(L):
        w = out[off[f"w{l}"]:off[f"w{l}"] + C * C * 9].reshape(C, C, 3, 3)
        w *= g_res
        w[:5] *= ST_TRUNK_LEAK
    head = out[off["head_w"]:off["head_w"] + nh * C].reshape(nh, C)
    head[0] = 0.0
    head[0, 0] = 1.0
    head[1] = 0.0
    head[1, 1], head[1, 2] = ST_XY_GAIN, -ST_XY_GAIN
    head[2] = 0.0
    head[2, 3], head[2, 4] = ST_XY_GAIN, -ST_XY_GAIN
    head[3:] *= 0.3
    return out.astype(np.float32)


def make_weights(cfg: Config, flavour: Optional[str] = None, seed: Optional[int] = None,
                 calibration: Optional[dict] = None) -> np.ndarray:
    """Final fp32 blob for `cfg`.  `flavour` defaults to "literal" for cfg 0, "lc" otherwise."""
    net = cfg.net
    seed = cfg.weight_seed if seed is None else int(seed)
    if flavour is None:
        flavour = "literal" if cfg.index == 0 else "lc"
    blob = he_normal_blob(net, seed)
    if flavour == "literal":
        return blob
    if flavour == "base":          # g_res only; what the calibration script starts from
        return apply_recipe(net, blob, cfg.g_res, [1.0] * net.head_channels, 1.0, 0.0)
    if flavour == "st_base":
        return st_base_blob(net, seed, cfg.g_res, cfg.frames.sigma_px)
    cal = load_calibration() if calibration is None else calibration
    key = calibration_key(cfg, flavour, seed)
    if key not in cal:
        raise KeyError(f"no calibration entry {key!r}; run tests/golden/make_calibration.py")
    e = cal[key]
    if flavour == "st":
        out = st_base_blob(net, seed, cfg.g_res, cfg.frames.sigma_px).astype(np.float64)
        off = blob_offsets(net)
        out[off["head_w"]:off["head_w"] + net.channels] *= float(e["kappa"])
        out[off["head_b"]] = float(e["b_p"])
        return out.astype(np.float32)
    return apply_recipe(net, blob, cfg.g_res, e["row_gain"], e["kappa"], e["b_p"])


def dloc_he_normal_blob(spec, seed: int, head_gain: float = 1.0, p_bias: float = 0.0) -> np.ndarray:
    """He-normal weights (std = sqrt(2 / fan_in)) and zero biases for a DlocSpec, in blob order
    (smlm.h: DilatedLoc topology); the head rows are scaled by head_gain and the detection bias
    set to p_bias (input choices, like kappa / b_p of the residual nets)."""
    rng = np.random.default_rng([int(seed), 0xD10C])
    parts = []
    for name, co, ci, k in spec.layers():
        w = rng.normal(0.0, np.sqrt(2.0 / (ci * k * k)), size=co * ci * k * k)
        b = np.zeros(co)
        if name == "head":
            w *= head_gain
            b[0] = p_bias
        parts += [w, b]
    blob = np.concatenate(parts).astype(np.float32)
    assert blob.size == spec.n_params()
    return blob
