"""B200-native (sm_100a) hot path of arXiv 2410.02314: DilatedLoc-style inference over stacks
of single-molecule frames plus on-GPU post-processing, as a C-ABI library
(include/smlm.h) with a thin ctypes binding.  See DESIGN.md."""
from .binding import (ABI_VERSION, BF16, CONV_AUTO, CONV_DIRECT, CONV_TCGEN05, EMITTER_DTYPE,
                      ERR_CUDA, ERR_INVALID_ARG, ERR_OOM, ERR_OVERFLOW, ERR_UNSUPPORTED_DEVICE,
                      EXPORTS, FP16, FP32, TILE_MERGE_NONE, TILE_MERGE_ROW, FUSE_ALL, FUSE_AUTO, FUSE_HEAD, FUSE_NONE, FUSE_PAIRS_1CTA, STEM_AUTO, STEM_CUDA_CORES, STEM_TENSOR, KERNEL_CONV, KERNEL_CONV_PAIR, KERNEL_POST, KERNEL_STEM, OK, CameraParams, Localizer, NetDesc, Ring, SmlmError,
                      desc_from_spec, emitters_to_numpy, lib, make_desc, PostParams, postprocess_static, debug_fill,
                      POST_STATIC_MAX_TILES, POST_STATIC_SCRATCH_BYTES)

from .dloc_binding import (DLOC_EMITTER_DTYPE, DLOC_EXPORTS, DLOC_HEADS, DlocDesc, DlocLocalizer, dloc_desc,
                           dloc_desc_from_spec, dloc_emitters_to_numpy)

__all__ = ["DLOC_EMITTER_DTYPE", "DLOC_EXPORTS", "DLOC_HEADS", "DlocDesc", "DlocLocalizer", "dloc_desc",
           "dloc_desc_from_spec", "dloc_emitters_to_numpy",
           "ABI_VERSION", "BF16", "CONV_AUTO", "CONV_DIRECT", "CONV_TCGEN05", "EMITTER_DTYPE",
           "ERR_CUDA", "ERR_INVALID_ARG", "ERR_OOM", "ERR_OVERFLOW", "ERR_UNSUPPORTED_DEVICE",
           "EXPORTS", "FP16", "FP32", "TILE_MERGE_NONE", "TILE_MERGE_ROW", "FUSE_ALL", "FUSE_AUTO", "FUSE_HEAD", "FUSE_NONE", "FUSE_PAIRS_1CTA", "STEM_AUTO", "STEM_CUDA_CORES", "STEM_TENSOR", "KERNEL_CONV", "KERNEL_CONV_PAIR", "KERNEL_POST", "KERNEL_STEM", "OK", "CameraParams", "Localizer", "NetDesc", "Ring", "SmlmError",
           "desc_from_spec", "emitters_to_numpy", "lib", "make_desc", "PostParams", "postprocess_static", "debug_fill",
           "POST_STATIC_MAX_TILES", "POST_STATIC_SCRATCH_BYTES"]
