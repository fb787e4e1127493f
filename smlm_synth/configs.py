"""Workload table: the five BASELINE.json configs as plain data.

This module holds NO arithmetic of the method (no convolution, no activation, no
detection rule).  It only names sizes, so that the oracle tests, the CUDA tests and
bench.py all ask the generators for the same thing.

Sources: BASELINE.json `configs[0..4]`; SURVEY.md section 8(a) size table and 8(d)
input table; readings G6, G12, G18, G20 (restated in DESIGN.md).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Tuple


@dataclass(frozen=True)
class NetSpec:
    channels: int                 # C
    dilations: Tuple[int, ...]    # d_l, l = 0..L-1
    head_channels: int            # 5: p,dx,dy,N,bg   6: p,dx,dy,z,N,bg
    precision: str                # "fp32" | "bf16" | "fp16" (fp16: the 8(f)-4 activation-precision variant)
    stem_relu: int = 1            # reading G3
    norm_scale: float = 1000.0    # BASELINE.json configs[0]: (x-100)/1000
    xy_scale: float = 0.5         # tanh*0.5
    z_scale_nm: float = 700.0     # reading G6
    photon_scale: float = 1000.0  # reading G6
    bg_scale: float = 100.0       # reading G6
    in_frames: int = 1            # 3: temporal context, frames f-1, f, f+1 as stem input channels (G24)

    @property
    def n_layers(self) -> int:
        return len(self.dilations)

    @property
    def radius(self) -> int:
        """Receptive-field radius of the maps: 1 (stem) + sum of dilations."""
        return 1 + sum(self.dilations)

    def n_params(self) -> int:
        C, L, nh = self.channels, self.n_layers, self.head_channels
        return (C * self.in_frames * 9 + C) + L * (C * C * 9 + C) + (nh * C + nh)

    def flop_per_px(self) -> int:
        """2 x MAC: stem 18C, each layer 18C^2, head 2C n_h."""
        C, L, nh = self.channels, self.n_layers, self.head_channels
        return 18 * C * self.in_frames + 18 * C * C * L + 2 * C * nh


@dataclass(frozen=True)
class DlocSpec:
    """The paper's own topology: DCD dense blocks of dilated
    convolutions, a two-stage U-Net, DECODE-style heads with uncertainties.  The paper gives no
    widths: every number here is a reading (D1-D9)."""
    c0: int = 48                                  # base width (D1)
    growth: int = 16                              # channels per DCD layer (D1)
    n_blocks: int = 4                             # 1 coarse-grained + 3 multi-scale
    dilations: Tuple[int, ...] = (2, 4, 8, 16)
    in_frames: int = 1                            # 3: frames f-1, f, f+1 (D8)
    precision: str = "fp32"
    stem_relu: int = 1
    norm_scale: float = 1000.0
    xy_scale: float = 0.5
    z_scale_nm: float = 700.0
    photon_scale: float = 1000.0
    bg_scale: float = 100.0
    sigma_xy_px: float = 3.0                      # D7
    sigma_z_nm: float = 700.0
    sigma_photons: float = 1000.0
    head_channels: int = 10

    def layers(self):
        """(name, c_out, c_in, k) of every convolution in blob order."""
        C, G = self.c0, self.growth
        out = [("stem", C, self.in_frames, 3)]
        for b in range(self.n_blocks):
            for i in range(len(self.dilations)):
                out.append((f"b{b}l{i}", G, C + i * G, 3))
            out.append((f"b{b}t", C, C + len(self.dilations) * G, 1))
        out += [("enc1", 2 * C, C, 3), ("enc2", 4 * C, 2 * C, 3), ("dec1", 2 * C, 6 * C, 3), ("dec0", C, 3 * C, 3),
                ("head", self.head_channels, C, 1)]
        return out

    def n_params(self) -> int:
        return sum(co * ci * k * k + co for _, co, ci, k in self.layers())


@dataclass(frozen=True)
class FrameSpec:
    n_frames: int
    height: int
    width: int
    emitters_per_frame: int       # reading G18: round(density x area)
    photons: Tuple[float, float]  # uniform range
    background: Tuple[float, float]
    sigma_px: float = 1.3
    astigmatic: bool = False      # cfg 2: sigma_x(z), sigma_y(z)
    z_range_nm: Tuple[float, float] = (0.0, 0.0)
    offset: float = 100.0
    gain: float = 1.0
    camera_maps: bool = False     # cfg 3: per-pixel offset ~ N(100,2), gain ~ N(2.0,0.1)
    pixel_size_nm: float = 100.0


@dataclass(frozen=True)
class Config:
    index: int
    name: str
    frames: FrameSpec
    net: NetSpec
    threshold: float = 0.3
    tile: int = 0                 # cfg 3: 512
    writeback_batch: int = 0      # cfg 4: 256
    g_res: float = 1.0            # reading G12: trunk gain (1/sqrt(L) for L = 12)
    oracle_frames: int = 8        # SURVEY.md 8(d) "oracle subset n_o"
    weight_seed: int = 7
    frame_seed: int = 2410


_D12 = (1, 2, 4, 8) * 3

CONFIGS = {
    0: Config(0, "cfg0_tiny2d_fp32",
              FrameSpec(8, 64, 64, 10, (1000.0, 5000.0), (50.0, 200.0)),
              NetSpec(16, (1, 2, 4, 8), 5, "fp32"),
              g_res=1.0, oracle_frames=8),
    1: Config(1, "cfg1_2d_256_bf16",
              FrameSpec(1000, 256, 256, 655, (1000.0, 5000.0), (50.0, 200.0)),
              NetSpec(48, _D12, 5, "bf16"),
              g_res=12 ** -0.5, oracle_frames=8),
    2: Config(2, "cfg2_3d_astig_512_bf16",
              FrameSpec(2000, 512, 512, 3932, (2000.0, 8000.0), (50.0, 200.0),
                        astigmatic=True, z_range_nm=(-700.0, 700.0)),
              NetSpec(64, _D12, 6, "bf16"),
              g_res=12 ** -0.5, oracle_frames=2),
    3: Config(3, "cfg3_fov2048_tiled_bf16",
              FrameSpec(500, 2048, 2048, 41943, (1000.0, 5000.0), (50.0, 200.0),
                        offset=100.0, gain=2.0, camera_maps=True),
              NetSpec(48, _D12, 5, "bf16"),
              tile=512, g_res=12 ** -0.5, oracle_frames=1),
    4: Config(4, "cfg4_dense_stream_bf16",
              FrameSpec(10000, 256, 256, 2621, (500.0, 3000.0), (100.0, 300.0)),
              NetSpec(48, _D12, 5, "bf16"),
              writeback_batch=256, g_res=12 ** -0.5, oracle_frames=8),
}


def get_config(i: int) -> Config:
    return CONFIGS[int(i)]
