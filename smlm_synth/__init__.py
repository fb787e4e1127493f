"""Seeded synthetic inputs shared by the oracle tests, the CUDA tests and bench.py.

Holds none of the method's arithmetic: it draws frames and weights and nothing else.
"""
from .configs import CONFIGS, Config, DlocSpec, FrameSpec, NetSpec, get_config
from .frames import FrameStack, camera_maps, make_frames
from .weights import (apply_recipe, blob_offsets, blob_size, calibration_key, dloc_he_normal_blob,
                      he_normal_blob, load_calibration, make_weights)

__all__ = ["CONFIGS", "Config", "DlocSpec", "dloc_he_normal_blob", "FrameSpec", "NetSpec", "get_config", "FrameStack",
           "camera_maps", "make_frames", "apply_recipe", "blob_offsets", "blob_size",
           "calibration_key", "he_normal_blob", "load_calibration", "make_weights"]
