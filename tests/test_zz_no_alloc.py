"""smlm_postprocess_static: the one entry point of the library that allocates nothing.

It is for programs that cannot let a library call cudaMalloc under them: an acquisition loop
that must not stall the device while camera frames stream in, a plug-in inside a host program
that owns all GPU memory, a process that may only allocate at start-up (include/smlm.h has the
full text).  Its compaction bookkeeping lives in a fixed 1 MiB array inside the library's
device code, shared by every call on a device and never cleared, so these tests make two calls
in a row - the second on different input - and compare each with the ctx path
(smlm_debug_postprocess, which allocates) record by record, at the tolerances of
test_gpu_parity.py's post-processing tests.

The file name sorts after every other test file on purpose: the suite runs with `pytest -x`, and a
failure here must not hide the parity tests.  The tests build all their inputs themselves, so
they pass alone in a fresh process and after the rest of the suite.
"""
import ctypes as C
import os
import subprocess
import tempfile

import numpy as np
import pytest

from smlm_synth import NetSpec
import paper_2410_02314_b200 as P
from paper_2410_02314_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FLOAT_TOL = (("x_nm", 1e-6), ("y_nm", 1e-6), ("z_nm", 1e-5), ("photons", 1e-5), ("bg", 1e-5), ("p", 1e-5))
TH, TW = 32, 64   # the tile of the fixed output order (smlm.h)


# ------------------------------------------------------------------ host side (no GPU needed)
def test_post_params_layout_and_limits_match_header():
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "smlm.h"
int main(void) {
  printf("%zu %zu %zu %d %d\n", sizeof(smlm_post_params), offsetof(smlm_post_params, xy_scale),
         offsetof(smlm_post_params, pixel_size_nm), SMLM_POST_STATIC_SCRATCH_BYTES, SMLM_POST_STATIC_MAX_TILES);
  return 0;
}
'''
    with tempfile.TemporaryDirectory() as d:
        src, exe = os.path.join(d, "t.c"), os.path.join(d, "t")
        open(src, "w").write(prog)
        subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), src, "-o", exe], check=True)
        got = [int(v) for v in subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()]
    PP = binding.PostParams
    assert got == [C.sizeof(PP), PP.xy_scale.offset, PP.pixel_size_nm.offset, binding.POST_STATIC_SCRATCH_BYTES,
                   binding.POST_STATIC_MAX_TILES]
    assert 256 + 4 * binding.POST_STATIC_MAX_TILES == binding.POST_STATIC_SCRATCH_BYTES


def test_oversized_and_malformed_calls_are_refused_before_any_gpu_work():
    """The argument checks come before the first CUDA call, so they can be exercised anywhere.
    The pointers are never dereferenced on the host; 4096 stands in for an aligned address."""
    fake = 4096
    per_frame = ((256 + TH - 1) // TH) * ((256 + TW - 1) // TW)          # 32 tiles per 256 x 256 frame
    fits = binding.POST_STATIC_MAX_TILES // per_frame
    with pytest.raises(P.SmlmError) as ei:
        binding.postprocess_static(fake, 5, 0.5, fake, 16, fake, shape=(fits + 1, 256, 256), stream=0)
    assert ei.value.status == P.ERR_INVALID_ARG
    msg = str(ei.value)
    assert "SMLM_POST_STATIC_MAX_TILES" in msg and str(binding.POST_STATIC_MAX_TILES) in msg and str(fits) in msg
    for kw in (dict(maps=None, shape=(1, 8, 8)), dict(shape=(1, 0, 8)), dict(shape=(-1, 8, 8)), dict(heads=4),
               dict(out=fake + 8), dict(cnt=None), dict(cap=-1)):
        with pytest.raises(P.SmlmError) as ei:
            binding.postprocess_static(kw.get("maps", fake), kw.get("heads", 5), 0.5, kw.get("out", fake),
                                       kw.get("cap", 16), kw.get("cnt", fake), shape=kw.get("shape", (1, 8, 8)),
                                       stream=0)
        assert ei.value.status == P.ERR_INVALID_ARG and len(str(ei.value)) > 20, kw


# ------------------------------------------------------------------ on the GPU
def _maps(seed, n, nh, H, W):
    rng = np.random.default_rng(seed)
    o = rng.normal(0, 1.0, size=(n, nh, H, W))
    o[:, 0] = np.round(rng.normal(0, 1.5, size=(n, H, W)) * 2) / 2        # many exact ties
    return o.astype(np.float32)


def _ctx_path(torch, o, nh, thr, cap):
    """The existing path: smlm_debug_postprocess on a ctx (sorted by (frame, pix))."""
    spec = NetSpec(16, (1,), nh, "fp32")
    with P.Localizer(P.desc_from_spec(spec), np.zeros(spec.n_params(), np.float32)) as loc:
        maps = torch.from_numpy(o).cuda()
        buf = torch.zeros(max(cap, 1) * 32, dtype=torch.uint8, device="cuda")
        cnt = loc.postprocess(maps, loc.camera(100.0, 100.0, 1.0), thr, buf, cap)
        torch.cuda.synchronize()
        return P.emitters_to_numpy(buf, min(cnt.value, cap)), int(cnt.value)


def _static_path(torch, o, nh, thr, cap, fill=0xAB):
    """The no-allocation path -> (records in the order the GPU wrote them, count)."""
    maps = torch.from_numpy(o).cuda()
    buf = torch.full((max(cap, 1) * 32,), fill, dtype=torch.uint8, device="cuda")
    cnt = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    binding.postprocess_static(maps, nh, thr, buf, cap, cnt)
    torch.cuda.synchronize()
    found = int(cnt.item())
    raw = buf.cpu().numpy()[: min(found, cap) * 32].copy()
    return raw.view(P.EMITTER_DTYPE), found


def _tile_order_key(em, H, W):
    y, x = em["pix"] // W, em["pix"] % W
    return np.stack([em["frame"], y // TH, x // TW, y % TH, x % TW], axis=1)


def _assert_same(em_s, found_s, em_c, found_c, H, W):
    assert found_s == found_c
    key = _tile_order_key(em_s, H, W)
    assert all(tuple(key[i]) < tuple(key[i + 1]) for i in range(len(key) - 1)), "documented list order"
    srt = em_s[np.lexsort((em_s["pix"], em_s["frame"]))]
    assert np.array_equal(srt["frame"], em_c["frame"]) and np.array_equal(srt["pix"], em_c["pix"])
    for k, rel in FLOAT_TOL:
        np.testing.assert_allclose(srt[k], em_c[k], rtol=rel, atol=1e-4, err_msg=k)


@pytest.mark.gpu
def test_static_path_equals_ctx_path_on_two_calls_in_a_row():
    import torch
    # call 1: three ragged frames (3 x 3 tiles each), six heads; call 2 right behind it on a
    # larger, different problem with five heads: whatever call 1 left in the scratch array must
    # not show; call 3 = call 1 again: the list is byte-identical (fixed order).
    cases = [(11, 3, 6, 75, 133, 0.3), (12, 5, 5, 160, 200, 0.6), (11, 3, 6, 75, 133, 0.3)]
    lists = []
    for seed, n, nh, H, W, thr in cases:
        o = _maps(seed, n, nh, H, W)
        cap = n * ((H + 1) // 2) * ((W + 1) // 2)
        em_s, found_s = _static_path(torch, o, nh, thr, cap)
        em_c, found_c = _ctx_path(torch, o, nh, thr, cap)
        assert found_c > 50 * n
        _assert_same(em_s, found_s, em_c, found_c, H, W)
        lists.append(em_s.tobytes())
    assert lists[0] == lists[2]


@pytest.mark.gpu
def test_static_path_thresholds_overflow_and_empty_calls():
    import torch
    n, nh, H, W = 2, 5, 70, 150
    o = _maps(21, n, nh, H, W)
    cap = n * ((H + 1) // 2) * ((W + 1) // 2)
    full, found = _static_path(torch, o, nh, 0.4, cap)
    for thr in (-1.0, 0.0, 0.7, 1.0, 2.0):                             # every maximum ... none
        em_s, found_s = _static_path(torch, o, nh, thr, cap)
        em_c, found_c = _ctx_path(torch, o, nh, thr, cap)
        _assert_same(em_s, found_s, em_c, found_c, H, W)
    # overflow: the count is the true one, the stored records are the head of the full list,
    # and nothing is written behind them
    small = found // 3
    maps = torch.from_numpy(o).cuda()
    buf = torch.full(((small + 4) * 32,), 0xCD, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    binding.postprocess_static(maps, nh, 0.4, buf, small, cnt)
    torch.cuda.synchronize()
    raw = buf.cpu().numpy()
    assert int(cnt.item()) == found > small
    assert raw[: small * 32].tobytes() == full[:small].tobytes() and (raw[small * 32:] == 0xCD).all()
    # count only (no list), and an empty call: the count is still written
    binding.postprocess_static(maps, nh, 0.4, None, 0, cnt)
    torch.cuda.synchronize()
    assert int(cnt.item()) == found
    binding.postprocess_static(None, nh, 0.4, None, 0, cnt, shape=(0, H, W))
    torch.cuda.synchronize()
    assert int(cnt.item()) == 0
    # and the array still serves the next ordinary call
    em_s, found_s = _static_path(torch, o, nh, 0.4, cap)
    assert found_s == found and em_s.tobytes() == full.tobytes()
