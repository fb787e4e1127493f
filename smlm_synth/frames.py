"""Seeded synthetic single-molecule frames (inputs only; no arithmetic of the method).

Stand-in for the paper's own data (simulations derived from a public challenge set and
200 000 random-dot 128x128 frames), which are not available and
are not recreated.  Shapes and statistics follow BASELINE.json `configs`; readings
G18-G21 of SURVEY.md 8(c) (restated in DESIGN.md "Input recipe"):

  G18  fixed emitter count per frame, positions U[-1/2, W-1/2) x U[-1/2, H-1/2)
       (pixel centres at integer coordinates, reading G7)
  G19  pixel-integrated Gaussian PSF:
       lam(y,x) = bg + sum_e N_e * dE_x * dE_y,
       dE_x = 1/2 [erf((x+1/2-x_e)/(sqrt2 s_x)) - erf((x-1/2-x_e)/(sqrt2 s_x))]
       cfg 2: s_x = 1.3 sqrt(1+((z-250)/400)^2), s_y = 1.3 sqrt(1+((z+250)/400)^2)
  G20  background: one scalar per frame, uniform
  G21  adu = clamp(floor(Poisson(lam) * gain + offset + 1/2), 0, 65535); no read noise;
       cfg 3: offset_map ~ N(100, 2), gain_map ~ N(2.0, 0.1) clipped to >= 0.5

Every frame f has its own generator seeded with (frame_seed, cfg index, f), so any
subset of frames can be produced independently and is identical on every machine.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np
from scipy.special import erf

from .configs import Config, FrameSpec

_SQRT2 = np.sqrt(2.0)


@dataclass
class FrameStack:
    frames: np.ndarray                  # uint16 [n][H][W]
    offset_map: Optional[np.ndarray]    # float32 [H][W] or None
    gain_map: Optional[np.ndarray]      # float32 [H][W] or None
    offset: float
    gain: float
    pixel_size_nm: float
    truth: list                         # per frame: float64 [E][5] = x_px, y_px, z_nm, photons, bg


def camera_maps(cfg: Config):
    """Per-pixel offset/gain maps for cfg 3 (None, None otherwise).  Fixed per config."""
    fs = cfg.frames
    if not fs.camera_maps:
        return None, None
    rng = np.random.default_rng([cfg.frame_seed, cfg.index, 0x0CA3])
    off = rng.normal(100.0, 2.0, size=(fs.height, fs.width))
    gain = np.clip(rng.normal(2.0, 0.1, size=(fs.height, fs.width)), 0.5, None)
    return off.astype(np.float32), gain.astype(np.float32)


def _sigmas(fs: FrameSpec, z: np.ndarray):
    if fs.astigmatic:
        sx = fs.sigma_px * np.sqrt(1.0 + ((z - 250.0) / 400.0) ** 2)
        sy = fs.sigma_px * np.sqrt(1.0 + ((z + 250.0) / 400.0) ** 2)
    else:
        sx = np.full_like(z, fs.sigma_px)
        sy = np.full_like(z, fs.sigma_px)
    return sx, sy


def expected_photons(fs: FrameSpec, xe, ye, ze, ne, bg, H=None, W=None) -> np.ndarray:
    """lam(y,x) of reading G19 for one frame, float64 [H][W]."""
    H = fs.height if H is None else H
    W = fs.width if W is None else W
    lam = np.full(H * W, float(bg))
    E = len(xe)
    if E == 0:
        return lam.reshape(H, W)
    sx, sy = _sigmas(fs, ze)
    half = int(np.ceil(5.0 * max(sx.max(), sy.max()))) + 1
    k = np.arange(-half, half + 1)                       # patch offsets
    cx = np.rint(xe).astype(np.int64)
    cy = np.rint(ye).astype(np.int64)
    px = cx[:, None] + k[None, :]                        # [E][P] absolute pixel columns
    py = cy[:, None] + k[None, :]
    ex = 0.5 * (erf((px + 0.5 - xe[:, None]) / (_SQRT2 * sx[:, None]))
                - erf((px - 0.5 - xe[:, None]) / (_SQRT2 * sx[:, None])))
    ey = 0.5 * (erf((py + 0.5 - ye[:, None]) / (_SQRT2 * sy[:, None]))
                - erf((py - 0.5 - ye[:, None]) / (_SQRT2 * sy[:, None])))
    ex = np.where((px >= 0) & (px < W), ex, 0.0)
    ey = np.where((py >= 0) & (py < H), ey, 0.0)
    chunk = max(1, 2_000_000 // (len(k) * len(k)))
    for s in range(0, E, chunk):
        e = slice(s, s + chunk)
        patch = ne[e, None, None] * ey[e, :, None] * ex[e, None, :]
        idx = np.clip(py[e], 0, H - 1)[:, :, None] * W + np.clip(px[e], 0, W - 1)[:, None, :]
        lam += np.bincount(idx.ravel(), weights=patch.ravel(), minlength=H * W)
    return lam.reshape(H, W)


def make_frames(cfg: Config, n: Optional[int] = None, first: int = 0,
                height: Optional[int] = None, width: Optional[int] = None,
                emitters: Optional[int] = None) -> FrameStack:
    """Frames first .. first+n-1 of config `cfg`.

    `height`/`width`/`emitters` override the config's frame size (used for crops and
    ragged-size parity cases); the emitter count then scales with the area unless given.
    """
    fs = cfg.frames
    n = fs.n_frames if n is None else int(n)
    H = fs.height if height is None else int(height)
    W = fs.width if width is None else int(width)
    if emitters is None:
        E = fs.emitters_per_frame
        if (H, W) != (fs.height, fs.width):
            E = int(round(E * (H * W) / float(fs.height * fs.width)))
    else:
        E = int(emitters)
    off_map, gain_map = camera_maps(cfg)
    if off_map is not None and (H, W) != (fs.height, fs.width):
        off_map = np.ascontiguousarray(off_map[:H, :W])
        gain_map = np.ascontiguousarray(gain_map[:H, :W])
    out = np.empty((n, H, W), dtype=np.uint16)
    truth = []
    for i in range(n):
        f = first + i
        rng = np.random.default_rng([cfg.frame_seed, cfg.index, 1, f])
        xe = rng.uniform(-0.5, W - 0.5, size=E)
        ye = rng.uniform(-0.5, H - 0.5, size=E)
        ze = rng.uniform(fs.z_range_nm[0], fs.z_range_nm[1], size=E) if fs.astigmatic else np.zeros(E)
        ne = rng.uniform(fs.photons[0], fs.photons[1], size=E)
        bg = rng.uniform(fs.background[0], fs.background[1])
        lam = expected_photons(fs, xe, ye, ze, ne, bg, H, W)
        counts = rng.poisson(lam).astype(np.float64)
        g = gain_map.astype(np.float64) if gain_map is not None else fs.gain
        o = off_map.astype(np.float64) if off_map is not None else fs.offset
        adu = np.floor(counts * g + o + 0.5)
        out[i] = np.clip(adu, 0, 65535).astype(np.uint16)
        truth.append(np.stack([xe, ye, ze, ne, np.full(E, bg)], axis=1))
    return FrameStack(out, off_map, gain_map, fs.offset, fs.gain, fs.pixel_size_nm, truth)
