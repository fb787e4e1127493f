"""CPU-only checks of the boundary: the C-ABI library builds, loads, exports every function
include/smlm.h declares, its structs have the layout the ctypes binding assumes, and without
an sm_100 device it fails loudly (no CPU fallback)."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import numpy as np
import pytest

import paper_2410_02314_b200 as P
from paper_2410_02314_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "smlm.h")


def _declared_functions():
    src = open(HEADER, "r", encoding="utf-8").read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(smlm_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_function():
    lib = C.CDLL(build.build())
    names = _declared_functions()
    assert {"smlm_create", "smlm_localize", "smlm_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in smlm.h but not exported"
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and smlm.h disagree"


def test_dloc_header_exports_and_layout():
    """include/dloc.h: every declared function is exported; struct layouts match the binding."""
    lib = C.CDLL(build.build())
    src = open(os.path.join(ROOT, "include", "dloc.h"), "r", encoding="utf-8").read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = sorted(set(re.findall(r"\b(dloc_[a-z_0-9]+)\s*\(", src)))
    assert sorted(P.DLOC_EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in dloc.h but not exported"
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "dloc.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu\n", sizeof(dloc_net_desc), offsetof(dloc_net_desc, dilations),
         offsetof(dloc_net_desc, in_frames), offsetof(dloc_net_desc, sigma_xy_px), offsetof(dloc_net_desc, conv_impl),
         sizeof(dloc_emitter));
  return 0;
}
'''
    with tempfile.TemporaryDirectory() as d:
        src_c = os.path.join(d, "t.c")
        exe = os.path.join(d, "t")
        open(src_c, "w").write(prog)
        subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), src_c, "-o", exe], check=True)
        got = [int(v) for v in subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()]
    D = P.DlocDesc
    assert got == [C.sizeof(D), D.dilations.offset, D.in_frames.offset, D.sigma_xy_px.offset, D.conv_impl.offset,
                   P.DLOC_EMITTER_DTYPE.itemsize]


def test_struct_layout_matches_header():
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "smlm.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\n", sizeof(smlm_net_desc), offsetof(smlm_net_desc, dilations),
         offsetof(smlm_net_desc, head_channels), offsetof(smlm_net_desc, writeback_frames),
         offsetof(smlm_net_desc, fusion), offsetof(smlm_net_desc, in_frames), offsetof(smlm_net_desc, tile_merge),
         offsetof(smlm_net_desc, stem_impl),
         sizeof(smlm_camera_params), offsetof(smlm_camera_params, gain_map), sizeof(smlm_emitter),
         offsetof(smlm_emitter, p));
  return 0;
}
'''
    with tempfile.TemporaryDirectory() as d:
        src = os.path.join(d, "t.c")
        exe = os.path.join(d, "t")
        open(src, "w").write(prog)
        subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), src, "-o", exe], check=True)
        got = [int(v) for v in subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()]
    N, Cam = binding.NetDesc, binding.CameraParams
    want = [C.sizeof(N), N.dilations.offset, N.head_channels.offset, N.writeback_frames.offset,
            N.fusion.offset, N.in_frames.offset, N.tile_merge.offset, N.stem_impl.offset, C.sizeof(Cam), Cam.gain_map.offset, binding.EMITTER_DTYPE.itemsize,
            binding.EMITTER_DTYPE.fields["p"][1]]
    assert got == want
    assert binding.EMITTER_DTYPE.itemsize == 32


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    d = P.make_desc(channels=16, dilations=(1,), head_channels=5, precision=P.FP32)
    w = np.zeros(16 * 10 + (16 * 16 * 9 + 16) + 5 * 17, np.float32)
    with pytest.raises(P.SmlmError) as ei:
        P.Localizer(d, w)
    assert ei.value.status == P.ERR_UNSUPPORTED_DEVICE


def test_bad_descriptor_is_refused_before_touching_the_device():
    d = P.make_desc(channels=24, dilations=(1,), head_channels=5, precision=P.FP32)
    with pytest.raises(P.SmlmError) as ei:
        P.Localizer(d, np.zeros(24 * 10 + (24 * 24 * 9 + 24) + 5 * 25, np.float32))
    assert ei.value.status == P.ERR_INVALID_ARG
