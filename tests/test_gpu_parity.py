"""GPU parity tests: the CUDA library (through its C ABI) against the CPU oracle, element by
element on the same seeded inputs.

Tolerances (BASELINE.json north_star): raw output maps within 1e-4 (fp32 mode) / 2e-2 (bf16
mode) absolute; emitter count and pixel indices bit-exact outside the contested set;
sub-pixel coordinates within 0.02 px.
"""
import json
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from smlm_synth import NetSpec, get_config, make_frames, make_weights
import paper_2410_02314_b200 as P
import gpu_util as G

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
TOL = {"fp32": 1e-4, "bf16": 2e-2}
BF16_IMPLS = [pytest.param(P.CONV_DIRECT, id="direct"), pytest.param(P.CONV_TCGEN05, id="tcgen05")]


def _rand_blob(spec, seed, scale=0.25):
    rng = np.random.default_rng(seed)
    return rng.normal(0, scale, size=spec.n_params()).astype(np.float32)


# ------------------------------------------------------------------ cfg 0: fp32 reference mode
def test_cfg0_fp32_trunk_maps_and_emitters():
    cfg = get_config(0)
    fs = make_frames(cfg)
    w = make_weights(cfg)
    ck = G.cam_kwargs(fs)
    net, cam, o, dump = G.oracle_run("cfg0", cfg.net, w, fs.frames, ck, dump_trunk=True)
    og, tg = G.gpu_forward_maps(cfg.net, w, fs.frames, ck, dump_trunk=True)
    for l in range(cfg.net.n_layers + 1):
        assert np.max(np.abs(tg[:, l] - dump[:, l])) < 1e-4, f"trunk level {l}"
    assert np.max(np.abs(G.activated(cfg.net, og) - G.activated(cfg.net, o))) < 1e-4
    em_o = O.postprocess(net, o, cam, cfg.threshold)
    em_g = G.gpu_localize(cfg.net, w, fs.frames, ck, cfg.threshold)
    st = G.parity_gate(cfg.net, o, em_o, em_g, cfg.threshold, 1e-4, fs.pixel_size_nm, 64, 64)
    G.record("cfg0_fp32", gate=st)
    assert st["oracle"] > 50 and st["contested_frac"] < 0.5      # the gate is not vacuous
    assert st["rel_N"] < 1e-3 and st["rel_bg"] < 1e-3


# ------------------------------------------------------------------ post-processing alone
def _gpu_post(spec, o, threshold, pixel=100.0, capacity=None):
    torch = G.torch_mod()
    desc = P.desc_from_spec(spec)
    n, nh, H, W = o.shape
    cap = n * ((H + 1) // 2) * ((W + 1) // 2) if capacity is None else capacity
    with P.Localizer(desc, np.zeros(spec.n_params(), np.float32)) as loc:
        maps = torch.from_numpy(np.ascontiguousarray(o, dtype=np.float32)).cuda()
        buf = torch.zeros(max(cap, 1) * 32, dtype=torch.uint8, device="cuda")
        cnt = loc.postprocess(maps, loc.camera(pixel, 100.0, 1.0), threshold, buf, cap)
        torch.cuda.synchronize()
        return P.emitters_to_numpy(buf, min(cnt.value, cap)), int(cnt.value), loc.check()


with open(os.path.join(GOLDEN, "delta_maps.json"), "r", encoding="utf-8") as _fh:
    _DELTA = json.load(_fh)


@pytest.mark.parametrize("case", _DELTA["cases"], ids=[c["name"] for c in _DELTA["cases"]])
def test_postprocess_hand_placed_delta_maps(case):
    H, W = _DELTA["H"], _DELTA["W"]
    spec = NetSpec(16, (1,), 5, "fp32")
    o = np.zeros((1, 5, H, W))
    o[0, 0] = case["background_logit"]
    for s in case["spikes"]:
        logit = s["logit"] if "logit" in s else math.log(s["p"] / (1.0 - s["p"]))
        o[0, 0, s["y"], s["x"]] = logit
        for h, key in ((1, "o_dx"), (2, "o_dy"), (3, "o_N"), (4, "o_bg")):
            if key in s:
                o[0, h, s["y"], s["x"]] = s[key]
    em, found, status = _gpu_post(spec, o, case["threshold"], _DELTA["pixel_size_nm"])
    # fp32 maps: a spike placed within 1e-6 of the threshold in p is not representable
    exp = sorted(case["expect"], key=lambda e: e["pix"])
    assert status == P.OK
    assert [int(p) for p in em["pix"]] == [e["pix"] for e in exp], case["name"]
    for got, e in zip(em, exp):
        for key in ("x_nm", "y_nm", "p", "photons", "bg"):
            if key in e:
                assert float(got[key]) == pytest.approx(e[key], rel=2e-6, abs=1e-30), (case["name"], key)
        assert got["z_nm"] == 0.0


def test_postprocess_ties_thresholds_and_six_heads_match_oracle():
    rng = np.random.default_rng(42)
    H, W = 75, 133                                         # several tiles + ragged tail
    spec = NetSpec(16, (1,), 6, "fp32")
    net = O.net_from_spec(spec)
    cam = O.make_camera(100.0, 100.0, 1.0)
    o = rng.normal(0, 1.0, size=(3, 6, H, W))
    o[:, 0] = np.round(rng.normal(0, 1.5, size=(3, H, W)) * 2) / 2      # many exact ties
    o = o.astype(np.float32).astype(np.float64)
    for thr in (-1.0, 0.0, 0.3, 0.7, 1.0, 2.0):
        em_o = O.postprocess(net, o, cam, thr)
        em_g, found, status = _gpu_post(spec, o, thr)
        assert status == P.OK and found == len(em_o), thr
        assert np.array_equal(em_g["frame"], em_o["frame"]) and np.array_equal(em_g["pix"], em_o["pix"])
        if len(em_o):
            for k, rel in (("x_nm", 1e-6), ("y_nm", 1e-6), ("z_nm", 1e-5), ("photons", 1e-5), ("bg", 1e-5), ("p", 1e-5)):
                np.testing.assert_allclose(em_g[k], em_o[k], rtol=rel, atol=1e-4, err_msg=k)


def test_postprocess_saturation_and_overflow():
    spec = NetSpec(16, (1,), 5, "fp32")
    o = np.zeros((1, 5, 9, 9))
    o[0, 0] = -40.0
    o[0, 0, 4, 4] = 40.0
    o[0, 3, 4, 4] = 40.0
    o[0, 4, 4, 4] = -40.0
    em, found, status = _gpu_post(spec, o, 0.3)
    assert found == 1 and np.isfinite([em[k][0] for k in ("x_nm", "y_nm", "photons", "bg", "p")]).all()
    assert em["photons"][0] == pytest.approx(40000.0, rel=1e-6) and em["p"][0] == pytest.approx(1.0)
    # overflow: all-local-maxima on a checkerboard, capacity 3
    o = np.zeros((1, 5, 8, 8))
    o[0, 0, ::2, ::2] = 1.0
    em, found, status = _gpu_post(spec, o, 0.3, capacity=3)
    assert found == 16 and len(em) == 3 and status == P.ERR_OVERFLOW


# ------------------------------------------------------------------ ragged sizes, maps, 6 heads
@pytest.mark.parametrize("C,nh,H,W,dil", [(16, 5, 37, 41, (1, 2)), (32, 6, 70, 131, (1, 2, 4, 8)),
                                          (64, 6, 33, 200, (8, 4)), (48, 5, 130, 66, (2, 8, 1))])
def test_fp32_ragged_sizes_camera_maps(C, nh, H, W, dil):
    spec = NetSpec(C, dil, nh, "fp32")
    w = _rand_blob(spec, C + H, scale=0.12)
    rng = np.random.default_rng(H * W)
    frames = rng.integers(50, 4000, size=(3, H, W)).astype(np.uint16)
    offm = rng.normal(100, 2, size=(H, W)).astype(np.float32)
    gm = np.clip(rng.normal(2.0, 0.1, size=(H, W)), 0.5, None).astype(np.float32)
    ck = dict(pixel_size_nm=100.0, offset=0.0, gain=1.0, offset_map=offm, gain_map=gm)
    net, cam, o, dump = G.oracle_run(("ragged", C, H), spec, w, frames, ck, dump_trunk=True)
    og, tg = G.gpu_forward_maps(spec, w, frames, ck, dump_trunk=True)
    scale = max(1.0, float(np.abs(dump).max()))
    for l in range(spec.n_layers + 1):
        assert np.max(np.abs(tg[:, l] - dump[:, l])) < 1e-5 * scale, f"level {l}"
    assert np.max(np.abs(og - o)) < 2e-5 * scale
    em_o = O.postprocess(net, o, cam, 0.5)
    em_g = G.gpu_localize(spec, w, frames, ck, 0.5)
    st = G.parity_gate(spec, o, em_o, em_g, 0.5, 1e-4, 100.0, H, W)
    print("ragged gate", (C, nh, H, W), st)


# ------------------------------------------------------------------ cfg 1: hc (fp32 mode) and lc (bf16)
def test_cfg1_hc_weights_fp32_mode_index_gate():
    cfg = get_config(1)
    fs = make_frames(cfg, 2)
    w = make_weights(cfg, "hc")
    ck = G.cam_kwargs(fs)
    net, cam, o, _ = G.oracle_run("cfg1hc", cfg.net, w, fs.frames, ck)
    import dataclasses
    spec32 = dataclasses.replace(cfg.net, precision="fp32")
    og = G.gpu_forward_maps(spec32, w, fs.frames, ck)
    assert np.max(np.abs(G.activated(cfg.net, og) - G.activated(cfg.net, o))) < 1e-4
    em_o = O.postprocess(net, o, cam, cfg.threshold)
    em_g = G.gpu_localize(spec32, w, fs.frames, ck, cfg.threshold)
    st = G.parity_gate(cfg.net, o, em_o, em_g, cfg.threshold, 1e-4, fs.pixel_size_nm, 256, 256)
    G.record("cfg1_hc_fp32_mode", gate=st)
    assert st["oracle"] > 800 and st["contested_frac"] < 0.25 and st["flipped"] <= 4


def _bf16_maps_and_gate(name, cfg, fs, w, impl, H, W, max_contested, check_tol=True):
    """bf16 production precision: (1) every activated head map within 2e-2 of the oracle;
    (2) the index gate with the contested set built from 2 x the MEASURED p-map error of this
    run (gpu_util.parity_gate), its size bounded and recorded - the gate must not be vacuous."""
    ck = G.cam_kwargs(fs)
    net, cam, o, _ = G.oracle_run(name, cfg.net, w, fs.frames, ck)
    og = G.gpu_forward_maps(cfg.net, w, fs.frames, ck, conv_impl=impl)
    err = G.head_errors(cfg.net, o, og)
    if check_tol:
        assert err.max() < 2e-2, err
    dp = G.p_error(o, og)
    em_o = O.postprocess(net, o, cam, cfg.threshold)
    em_g = G.gpu_localize(cfg.net, w, fs.frames, ck, cfg.threshold, conv_impl=impl)
    st = G.parity_gate(cfg.net, o, em_o, em_g, cfg.threshold, 2e-2, fs.pixel_size_nm, H, W,
                       dp_measured=dp, check_tol=check_tol, o_gpu=og)
    impl_name = {P.CONV_DIRECT: "direct", P.CONV_TCGEN05: "tcgen05"}[impl]
    G.record(f"{name}_bf16_{impl_name}", gate=st, head_max_err=err, frames=len(fs.frames), H=H, W=W)
    if max_contested is not None:
        assert st["contested_frac_local"] <= max_contested, st
    assert st["uncontested_local"] >= 100, st
    return st


@pytest.mark.parametrize("impl", BF16_IMPLS)
def test_cfg1_lc_weights_bf16_maps_and_gate(impl):
    cfg = get_config(1)
    _bf16_maps_and_gate("cfg1lc", cfg, make_frames(cfg, 2), make_weights(cfg, "lc"), impl, 256, 256, 0.6)


@pytest.mark.parametrize("impl", BF16_IMPLS)
def test_cfg1_hc_weights_bf16_index_gate(impl):
    """The high-contrast p-head (logit std 3, the survey's strong index test) through the bf16
    kernels.  Its p-map error may exceed 2e-2 by construction (the logit error scales with the
    contrast), so the map tolerance is not asserted here; the index gate is, with
    the contested set from the measured error: no decision may differ outside it."""
    cfg = get_config(1)
    st = _bf16_maps_and_gate("cfg1hc", cfg, make_frames(cfg, 2), make_weights(cfg, "hc"), impl, 256, 256,
                             0.7, check_tol=False)
    assert st["oracle"] > 800


@pytest.mark.parametrize("impl", BF16_IMPLS)
def test_cfg2_crop_bf16_six_heads(impl):
    cfg = get_config(2)
    _bf16_maps_and_gate("cfg2crop", cfg, make_frames(cfg, 2, height=136, width=200), make_weights(cfg, "lc"),
                        impl, 136, 200, 0.6)


@pytest.mark.parametrize("impl", BF16_IMPLS)
def test_cfg4_dense_bf16(impl):
    """cfg 4 with the random `lc` weights: map parity, and the index gate outside the contested set.
    No cap on the contested fraction here (it is recorded: ~0.6 on this smooth p-map, DESIGN.md
    reading G28); the bounded index gate of cfg 4 is test_st_weights_bf16_index_gate."""
    cfg = get_config(4)
    _bf16_maps_and_gate("cfg4", cfg, make_frames(cfg, 1), make_weights(cfg, "lc"), impl, 256, 256, None)


@pytest.mark.parametrize("impl", BF16_IMPLS)
@pytest.mark.parametrize("ci", [1, 4])
def test_st_weights_bf16_index_gate(ci, impl):
    """The surrogate-trained weight set (smlm_synth "st", reading G28: sharp p-map peaks at the
    emitters, as P:61 describes the trained net's output) through the bf16 kernels: maps within
    2e-2, and the index gate must compare most detections bit-exactly - at most 15 % of the
    oracle's detections may lie in the contested set built from the measured local error."""
    cfg = get_config(ci)
    st = _bf16_maps_and_gate(f"cfg{ci}st", cfg, make_frames(cfg, 2), make_weights(cfg, "st"), impl, 256, 256, 0.15)
    assert st["oracle"] > 0.9 * 2 * min(cfg.frames.emitters_per_frame, 2621)


# ------------------------------------------------------------------ maps in the launch shape bench.py times
def _launch_shape_maps(name, cfg, fs, w, n, sample, tol=2e-2):
    """n frames cycling the distinct frames of fs through smlm_debug_forward_maps with the
    default micro-batch (cfg 1: 128 + 128 + tail views per launch): K2's work split - cluster /
    lane ranges of a few hundred rows that start and end mid-chain - is the one of the timed run.  Sampled
    frames are compared element by element with the oracle, and every frame with the first
    occurrence of the same distinct frame bit by bit (position in the launch must not matter)."""
    k = len(fs.frames)
    ck = G.cam_kwargs(fs)
    frames = np.ascontiguousarray(np.concatenate([fs.frames] * ((n + k - 1) // k))[:n])
    net, cam, o, _ = G.oracle_run(name, cfg.net, w, fs.frames, ck)
    og = G.gpu_forward_maps(cfg.net, w, frames, ck, conv_impl=P.CONV_TCGEN05)
    for f in range(k, n):
        assert np.array_equal(og[f], og[f % k]), f"frame {f} differs from frame {f % k}"
    errs = {}
    for f in sample:
        e = G.head_errors(cfg.net, o[f % k:f % k + 1], og[f:f + 1])
        assert e.max() < tol, (f, e)
        errs[str(f)] = e
    G.record(f"{name}_launch_shape_maps", frames=n, distinct=k, head_max_err=errs)


def test_cfg1_maps_in_timed_launch_shape_260_frames():
    cfg = get_config(1)     # default micro-batch: 128 + 128 + tail views per launch, layer pairs on 2-CTA clusters
    _launch_shape_maps("cfg1lc", cfg, make_frames(cfg, 2), make_weights(cfg, "lc"), 260, (0, 127, 128, 259))


def test_cfg2_maps_full_frame_in_multi_view_launch():
    cfg = get_config(2)
    _launch_shape_maps("cfg2full", cfg, make_frames(cfg, 1), make_weights(cfg, "lc"), 12, (0, 11))


def test_cfg3_tile_window_maps_in_multi_view_launch():
    """cfg 3 launches sets of 606 x 606 windows (512 + 2 x 47); the same window shape through
    the map export, 16 views per call, against the oracle on the same window."""
    cfg = get_config(3)
    fs = make_frames(cfg, 1, height=606, width=606)
    _launch_shape_maps("cfg3win", cfg, fs, make_weights(cfg, "lc"), 16, (0, 15))


# ------------------------------------------------------------------ bf16: tensor-core kernel vs CUDA-core kernel
@pytest.mark.parametrize("C,H,W,dil", [(48, 70, 300, (1, 2, 4, 8)), (64, 40, 129, (8, 1)),
                                       (16, 64, 64, (1, 2, 4, 8)), (32, 19, 517, (4, 2)),
                                       (16, 9, 9, (8, 4, 1)), (32, 3, 140, (2, 8)), (48, 1, 1, (1, 8))])
def test_tcgen05_matches_direct_bf16(C, H, W, dil):
    """Same rounding points (bf16 inputs and weights, fp32 accumulate, one RNE store), only the
    summation order differs: the stored bf16 maps may differ by an ulp here and there."""
    spec = NetSpec(C, dil, 5, "bf16")
    w = _rand_blob(spec, 100 + C, scale=(2.0 / (9 * C)) ** 0.5 * 0.6)
    rng = np.random.default_rng(W)
    frames = rng.integers(80, 3000, size=(3, H, W)).astype(np.uint16)
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    _, ta = G.gpu_forward_maps(spec, w, frames, ck, dump_trunk=True, conv_impl=P.CONV_DIRECT)
    _, tb = G.gpu_forward_maps(spec, w, frames, ck, dump_trunk=True, conv_impl=P.CONV_TCGEN05)
    assert np.array_equal(ta[:, 0], tb[:, 0])
    for l in range(1, spec.n_layers + 1):
        d = np.abs(ta[:, l] - tb[:, l])
        scale = np.maximum(np.abs(ta[:, l]), 1.0)
        assert np.max(d / scale) < 2.0 ** -6, f"level {l}: {np.max(d / scale)}"
        assert np.mean(d > 0) < 0.05, f"level {l}: {np.mean(d > 0)} of values differ"


# ------------------------------------------------------------------ tiling (cfg 3 mechanics)
@pytest.mark.parametrize("precision,impl", [("fp32", P.CONV_AUTO), ("bf16", P.CONV_DIRECT),
                                            ("bf16", P.CONV_TCGEN05)])
def test_tiled_equals_whole_frame(precision, impl):
    """cfg 3: tiles with a halo of radius+1, detections owned by the core tile.  The tiled
    result must equal whole-frame processing (bit-exact: the kernels' summation order does
    not depend on position) and hence the oracle, which never tiles."""
    spec = NetSpec(16, (1, 2, 4), 5, precision)                 # radius 8 -> halo 9
    w = _rand_blob(spec, 5, scale=0.2)
    rng = np.random.default_rng(77)
    H, W = 150, 173
    frames = rng.integers(80, 3000, size=(2, H, W)).astype(np.uint16)
    offm = rng.normal(100, 2, size=(H, W)).astype(np.float32)
    gm = np.clip(rng.normal(2.0, 0.1, size=(H, W)), 0.5, None).astype(np.float32)
    ck = dict(pixel_size_nm=100.0, offset=0.0, gain=1.0, offset_map=offm, gain_map=gm)
    whole = G.gpu_localize(spec, w, frames, ck, 0.5, conv_impl=impl)
    assert len(whole) > 100
    for tile, mb in ((64, 0), (64, 2), (40, 3), (128, 0)):
        tiled = G.gpu_localize(spec, w, frames, ck, 0.5, conv_impl=impl, tile=tile, micro_batch=mb)
        assert np.array_equal(tiled["frame"], whole["frame"]) and np.array_equal(tiled["pix"], whole["pix"]), tile
        for k in ("x_nm", "y_nm", "photons", "bg", "p"):
            assert np.array_equal(tiled[k], whole[k]), (tile, k)
    if precision == "fp32":
        net, cam, o, _ = G.oracle_run("tiled", spec, w, frames, ck)
        em_o = O.postprocess(net, o, cam, 0.5)
        G.parity_gate(spec, o, em_o, whole, 0.5, 1e-4, 100.0, H, W)


# ------------------------------------------------------------------ pipeline: ring, write-back, edge cases
def test_pinned_ring_and_writeback_batches_equal_device_path():
    cfg = get_config(0)
    fs = make_frames(cfg, 8)
    frames = np.concatenate([fs.frames] * 5)[:37]               # 37 frames, micro-batch 4 -> ragged tail
    w = make_weights(cfg)
    ck = G.cam_kwargs(fs)
    ref = G.gpu_localize(cfg.net, w, frames, ck, cfg.threshold, micro_batch=4)
    for kw in (dict(host_frames=True), dict(host_frames=True, host_out=True, writeback_frames=8),
               dict(host_out=True), dict(host_frames=True, host_out=True, writeback_frames=5, micro_batch=3)):
        kw.setdefault("micro_batch", 4)
        em = G.gpu_localize(cfg.net, w, frames, ck, cfg.threshold, **kw)
        assert np.array_equal(em, ref), kw
    # frames 8.. repeat frames 0..: same detections, shifted frame index
    a = ref[ref["frame"] < 8]
    b = ref[(ref["frame"] >= 8) & (ref["frame"] < 16)]
    assert np.array_equal(a["pix"], b["pix"]) and np.array_equal(a["frame"] + 8, b["frame"])


def test_writeback_every_frame_stress_equals_device_path():
    """A flush after every frame (writeback_frames = 1, micro_batch = 1): 600 flushes per call
    whose snapshots are written on the compute stream while earlier flushes may still run on
    the write-back stream.  The host list must equal the device-path list bit by bit."""
    cfg = get_config(0)
    fs = make_frames(cfg, 8)
    frames = np.ascontiguousarray(np.concatenate([fs.frames] * 75)[:600])
    w = make_weights(cfg)
    ck = G.cam_kwargs(fs)
    ref = G.gpu_localize(cfg.net, w, frames, ck, cfg.threshold, micro_batch=8)
    assert len(ref) > 10000
    for rep in range(20):
        em = G.gpu_localize(cfg.net, w, frames, ck, cfg.threshold, host_frames=True, host_out=True,
                            writeback_frames=1, micro_batch=1)
        assert np.array_equal(em, ref), rep


def test_edge_cases_empty_overflow_pageable_threshold():
    torch = G.torch_mod()
    cfg = get_config(0)
    fs = make_frames(cfg, 2)
    w = make_weights(cfg)
    ck = G.cam_kwargs(fs)
    em, found, status, _ = G.gpu_localize(cfg.net, w, fs.frames[:0], ck, 0.3, return_status=True)
    assert found == 0 and status == P.OK
    em, found, status, _ = G.gpu_localize(cfg.net, w, fs.frames, ck, 1.0, return_status=True)
    assert found == 0 and status == P.OK
    full = G.gpu_localize(cfg.net, w, fs.frames, ck, 0.3)
    em, found, status, _ = G.gpu_localize(cfg.net, w, fs.frames, ck, 0.3, capacity=5, return_status=True)
    assert found == len(full) and len(em) == 5 and status == P.ERR_OVERFLOW
    em, found, status, _ = G.gpu_localize(cfg.net, w, fs.frames, ck, 0.3, capacity=5, host_out=True,
                                          return_status=True)
    assert found == len(full) and len(em) == 5 and status == P.ERR_OVERFLOW
    allmax, n_all, status, _ = G.gpu_localize(cfg.net, w, fs.frames, ck, 0.0, return_status=True)
    assert status == P.OK and n_all >= len(full)
    assert {(int(f), int(q)) for f, q in zip(full["frame"], full["pix"])} <= \
           {(int(f), int(q)) for f, q in zip(allmax["frame"], allmax["pix"])}
    # pageable host frames are refused (they would silently serialise the copy)
    desc = P.desc_from_spec(cfg.net)
    with P.Localizer(desc, w) as loc:
        buf = torch.zeros(32 * 10, dtype=torch.uint8, device="cuda")
        with pytest.raises(P.SmlmError) as ei:
            loc.localize(torch.from_numpy(fs.frames.copy()), loc.camera(), 0.3, buf, 10)
        assert ei.value.status == P.ERR_INVALID_ARG
    # bad descriptors
    for kw in (dict(channels=24), dict(head_channels=4), dict(dilations=(17,)), dict(precision=7), dict(in_frames=2), dict(tile_merge=5)):
        base = dict(channels=16, dilations=(1,), head_channels=5, precision=P.FP32)
        base.update(kw)
        d = P.make_desc(**base)
        with pytest.raises(P.SmlmError) as ei:
            P.Localizer(d, np.zeros((d.channels * 10) + d.n_layers * (d.channels ** 2 * 9 + d.channels)
                                    + d.head_channels * (d.channels + 1), np.float32))
        assert ei.value.status == P.ERR_INVALID_ARG


# ------------------------------------------------------------------ production K3 (logit map from the last
# tcgen05 layer's epilogue + post_logits_kernel) against the oracle's rule, exactly
def _exact_post_check(spec, w, frames, ck, thr, **kw):
    """The production list must equal the ORACLE's post-processing applied to the GPU's own
    pre-activation maps (fp32 values are exact in fp64, so every comparison of the rule is
    decided identically): same (frame, pix) set with no contested-set allowance, decoded
    values to float rounding.  Pins the fused head (same bits as the debug maps), the 3x3
    test with its tie rule, ownership in tiled mode and the compaction."""
    net = O.net_from_spec(spec)
    cam = O.make_camera(**ck)
    og = G.gpu_forward_maps(spec, w, frames, ck, conv_impl=P.CONV_TCGEN05)
    em_o = O.postprocess(net, og.astype(np.float64), cam, thr)
    em_g = G.gpu_localize(spec, w, frames, ck, thr, conv_impl=P.CONV_TCGEN05, **kw)
    assert len(em_o) == len(em_g)
    assert np.array_equal(em_o["frame"], em_g["frame"]) and np.array_equal(em_o["pix"], em_g["pix"])
    for k, tol in (("x_nm", 2e-3), ("y_nm", 2e-3), ("z_nm", 2e-2), ("p", 1e-6)):      # + fp32 ulp of the value
        assert np.all(np.abs(em_o[k] - em_g[k]) <= tol + 2.4e-7 * np.abs(em_o[k])), k
    for k in ("photons", "bg"):
        assert np.max(np.abs(em_o[k] - em_g[k]) / np.maximum(np.abs(em_o[k]), 1.0), initial=0.0) <= 1e-5, k
    return len(em_o)


def test_production_post_equals_oracle_rule_on_gpu_maps_cfg1_and_cfg2_crop():
    cfg = get_config(1)
    fs = make_frames(cfg, 3)
    n = _exact_post_check(cfg.net, make_weights(cfg, "lc"), fs.frames, G.cam_kwargs(fs), cfg.threshold)
    assert n > 500
    cfg = get_config(2)
    fs = make_frames(cfg, 2, height=150, width=333)            # ragged, 6 heads, C = 64
    n = _exact_post_check(cfg.net, make_weights(cfg, "lc"), fs.frames, G.cam_kwargs(fs), cfg.threshold)
    assert n > 100
    n = _exact_post_check(cfg.net, make_weights(cfg, "lc"), fs.frames, G.cam_kwargs(fs), cfg.threshold,
                          tile=96, micro_batch=5)
    assert n > 100


def test_production_post_tie_rule_on_quantised_logits():
    """Logit = bf16(relu(xhat)) of a coarse integer image: thousands of exact ties between
    neighbours, plateaus, and image-border cases in the tcgen05 production path."""
    spec = NetSpec(16, (1,), 5, "bf16")
    C = 16
    w = np.zeros(spec.n_params(), np.float32)
    w[0 * 9 + 4] = 1.0                                         # stem channel 0 = centre tap
    off_head = C * 10 + (C * C * 9 + C)
    w[off_head + 0] = 1.0                                      # p head reads channel 0
    w[off_head + 1 * C + 1] = 0.3                              # dx head reads channel 1 (zero): dx = 0
    rng = np.random.default_rng(5)
    frames = (100 + 250 * rng.integers(0, 4, size=(3, 70, 150))).astype(np.uint16)   # 4 levels
    frames[1, 10:30, 20:60] = 1100                                                   # plateau
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    for thr in (0.3, 0.55, 0.0):
        n = _exact_post_check(spec, w, frames, ck, thr)
        assert n > 50 or thr == 0.55


# ------------------------------------------------------------------ fusion vs one kernel per step
@pytest.mark.parametrize("C,nh,H,W,dil,tile", [(48, 5, 70, 300, (1, 2, 4, 8), 0), (64, 6, 40, 129, (2, 8, 1), 0),
                                               (16, 5, 64, 64, (1,), 0), (32, 6, 19, 517, (4, 2), 0),
                                               (16, 5, 9, 9, (8, 4, 1), 0), (48, 5, 1, 1, (1, 8), 0),
                                               (48, 5, 150, 173, (1, 2, 4), 64)])
def test_fused_stem_and_heads_equal_unfused_bit_exact(C, nh, H, W, dil, tile):
    """SMLM_FUSE_ALL (K1 inside the first layer's kernel, K3's heads inside the last layer's
    epilogue) and SMLM_FUSE_AUTO (heads only) against SMLM_FUSE_NONE (stem_kernel, plain layers,
    heads from the stored map):
    same arithmetic and rounding points, so trunk levels and emitter records are identical
    bit by bit - with per-pixel camera maps, ragged sizes, H < d, 1x1 frames and tiles."""
    spec = NetSpec(C, dil, nh, "bf16")
    w = _rand_blob(spec, 300 + C + H, scale=(2.0 / (9 * C)) ** 0.5 * 0.6)
    off = C * 10 + len(dil) * (C * C * 9 + C)
    w[off + nh * C] = 0.2                                     # p-head bias: a usable detection rate
    rng = np.random.default_rng(H * 1000 + W)
    frames = rng.integers(80, 3000, size=(3, H, W)).astype(np.uint16)
    offm = rng.normal(100, 2, size=(H, W)).astype(np.float32)
    gm = np.clip(rng.normal(2.0, 0.1, size=(H, W)), 0.5, None).astype(np.float32)
    ck = dict(pixel_size_nm=100.0, offset=0.0, gain=1.0, offset_map=offm, gain_map=gm)
    kw = dict(conv_impl=P.CONV_TCGEN05)
    # SMLM_FUSE_ALL computes a_0 with the fmaf chain of stem.cu inside the first layer's kernel, so its
    # twin is the CUDA-core stem; the other modes share the default stem (tensor cores where it exists)
    cc = dict(stem_impl=P.STEM_CUDA_CORES, **kw)
    if not tile:
        ma, ta = G.gpu_forward_maps(spec, w, frames, ck, dump_trunk=True, fusion=P.FUSE_NONE, **cc)
        mb, tb = G.gpu_forward_maps(spec, w, frames, ck, dump_trunk=True, fusion=P.FUSE_ALL, **kw)
        assert np.array_equal(ta, tb) and np.array_equal(ma, mb)
    for thr in (0.5, 0.0):
        a = G.gpu_localize(spec, w, frames, ck, thr, fusion=P.FUSE_NONE, tile=tile, **cc)
        assert len(a) > 0 or H * W < 100
        b = G.gpu_localize(spec, w, frames, ck, thr, fusion=P.FUSE_ALL, tile=tile, **kw)
        assert len(a) == len(b) and a.tobytes() == b.tobytes(), (thr, "all")
        a = G.gpu_localize(spec, w, frames, ck, thr, fusion=P.FUSE_NONE, tile=tile, **kw)
        b = G.gpu_localize(spec, w, frames, ck, thr, fusion=P.FUSE_AUTO, tile=tile, **kw)
        assert len(a) == len(b) and a.tobytes() == b.tobytes(), (thr, "auto")


# ------------------------------------------------------------------ K1 on the tensor cores vs the CUDA-core stem
@pytest.mark.parametrize("C,prec,H,W,tile", [(48, "bf16", 70, 300, 0), (64, "bf16", 40, 129, 0), (16, "fp16", 33, 131, 0),
                                             (32, "bf16", 1, 1, 0), (48, "bf16", 150, 173, 64)])
def test_tensor_core_stem_equals_cuda_core_stem_to_rounding(C, prec, H, W, tile):
    """SMLM_STEM_TENSOR (three 16-bit pieces of every xhat and weight, fp32 accumulation in TMEM)
    against SMLM_STEM_CUDA_CORES (fp32 fmaf chain): a_0 is the same fp32 sum up to summation
    order, so after the one rounding to the storage type the two maps agree except for rare
    1-ulp flips - with per-pixel camera maps, ragged widths, 1x1 frames and tile windows."""
    spec = NetSpec(C, (1, 2), 5, prec)
    w = _rand_blob(spec, 900 + C + H, scale=(2.0 / (9 * C)) ** 0.5 * 0.6)
    w[C * 10 + 2 * (C * C * 9 + C) + 5 * C] = 0.2
    rng = np.random.default_rng(H * 77 + W)
    frames = rng.integers(80, 6000, size=(3, H, W)).astype(np.uint16)
    offm = rng.normal(100, 2, size=(H, W)).astype(np.float32)
    gm = np.clip(rng.normal(2.0, 0.1, size=(H, W)), 0.5, None).astype(np.float32)
    ck = dict(pixel_size_nm=100.0, offset=0.0, gain=1.0, offset_map=offm, gain_map=gm)
    kw = dict(conv_impl=P.CONV_TCGEN05)
    if not tile:
        _, ta = G.gpu_forward_maps(spec, w, frames, ck, dump_trunk=True, stem_impl=P.STEM_CUDA_CORES, **kw)
        _, tb = G.gpu_forward_maps(spec, w, frames, ck, dump_trunk=True, stem_impl=P.STEM_TENSOR, **kw)
        a0, b0 = ta[:, 0].astype(np.float64), tb[:, 0].astype(np.float64)
        ulp = 2.0 ** (-7 if prec == "bf16" else -10)         # one ulp of the storage type, relative, at the bottom of a binade
        rel = np.abs(a0 - b0) / np.maximum(np.abs(a0), 1e-3)
        assert rel.max() <= 1.01 * ulp, rel.max()                    # at most one ulp of the storage type
        assert np.mean(a0 != b0) < 0.02, np.mean(a0 != b0)           # and rarely
    a = G.gpu_localize(spec, w, frames, ck, 0.5, tile=tile, stem_impl=P.STEM_CUDA_CORES, **kw)
    b = G.gpu_localize(spec, w, frames, ck, 0.5, tile=tile, stem_impl=P.STEM_TENSOR, **kw)
    ka = {(int(f), int(q)) for f, q in zip(a["frame"], a["pix"])}
    kb = {(int(f), int(q)) for f, q in zip(b["frame"], b["pix"])}
    assert len(ka ^ kb) <= max(2, 0.02 * len(ka)), (len(ka), len(kb), len(ka ^ kb))


# ------------------------------------------------------------------ layer pairs (conv_pair.cu) vs one kernel per layer
@pytest.mark.parametrize("C,nh,n,H,W,dil,tile", [
    (48, 5, 5, 256, 256, (1, 2, 4, 8) * 3, 0),       # the cfg 1 trunk: six pairs, cluster of 2
    (48, 5, 3, 37, 130, (1, 2), 0),                  # ragged: 2 valid pixels in the second segment
    (32, 6, 2, 64, 100, (2, 4, 8, 16), 0),           # one segment (no neighbours), the paper's dilations
    (16, 5, 2, 21, 1000, (1, 2, 4, 8), 0),           # cluster of 8
    (48, 5, 2, 3, 17, (4, 8), 0),                    # H < d
    (48, 5, 1, 40, 1025, (1, 2), 0),                 # 9 segments: not a pair, must fall back
    (48, 5, 2, 300, 300, (4, 8, 1, 2, 4), 96),       # tiles (windows of 96 + halo), a single layer after the pairs
    (32, 5, 70, 24, 200, (1, 2, 4, 8), 0),           # more views than clusters x rows: several runs per cluster
    (16, 5, 48, 40, 300, (1, 2, 4, 8), 0),           # a full wave of 3-CTA clusters at C = 16 (one CTA per SM: TMEM)
    (32, 6, 40, 48, 512, (2, 4), 0)])                # a full wave of 4-CTA clusters (cta_group::2) at C = 32
def test_layer_pairs_equal_unfused_bit_exact(C, nh, n, H, W, dil, tile):
    """SMLM_FUSE_AUTO runs layers with dilations (d, 2d) as one kernel on a thread-block cluster
    (the map between them stays in shared memory, x halos exchanged through distributed shared
    memory).  Same operands, accumulation order and rounding points as one kernel per layer
    (SMLM_FUSE_HEAD), so head maps and emitter records must be identical bit by bit."""
    spec = NetSpec(C, dil, nh, "bf16")
    w = _rand_blob(spec, 700 + C + W, scale=(2.0 / (9 * C)) ** 0.5 * 0.6)
    off = C * 10 + len(dil) * (C * C * 9 + C)
    w[off + nh * C] = 0.2
    rng = np.random.default_rng(H * 1000 + W + 1)
    frames = rng.integers(80, 3000, size=(n, H, W)).astype(np.uint16)
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    kw = dict(conv_impl=P.CONV_TCGEN05)
    if not tile:
        ma = G.gpu_forward_maps(spec, w, frames, ck, fusion=P.FUSE_HEAD, **kw)
        for fusion in (P.FUSE_AUTO, P.FUSE_PAIRS_1CTA):
            mb = G.gpu_forward_maps(spec, w, frames, ck, fusion=fusion, **kw)
            assert np.array_equal(ma, mb), (fusion, float(np.max(np.abs(ma - mb))))
    for thr in (0.5, 0.0):
        a = G.gpu_localize(spec, w, frames, ck, thr, fusion=P.FUSE_HEAD, tile=tile, **kw)
        assert len(a) > 0
        for fusion in (P.FUSE_AUTO, P.FUSE_PAIRS_1CTA):     # cta_group::2 where the row has an even number of segments / ::1
            b = G.gpu_localize(spec, w, frames, ck, thr, fusion=fusion, tile=tile, **kw)
            assert len(a) == len(b) and a.tobytes() == b.tobytes(), (thr, fusion)


def test_layer_pairs_random_shapes_equal_unfused_bit_exact():
    """Seeded random shapes through the pair kernel (both cta_group variants) against one kernel
    per layer: widths on both sides of every segment boundary, heights around the dilations,
    every supported channel count, every (d, 2d) pair, with and without a trailing single layer."""
    rng = np.random.default_rng(20241002)
    for case in range(14):
        C = int(rng.choice([16, 32, 48]))
        d = int(rng.choice([1, 2, 4, 8]))
        dil = (d, 2 * d) + ((int(rng.choice([1, 2, 4])),) if rng.random() < 0.4 else ())
        seg = int(rng.integers(1, 6))
        W = int(np.clip(128 * seg + rng.integers(-3, 4), 1, 640))
        H = int(rng.choice([1, 2, d, 2 * d + 1, 3 * d + 2, 40]))
        n = int(rng.integers(1, 4))
        spec = NetSpec(C, dil, int(rng.choice([5, 6])), "bf16")
        w = _rand_blob(spec, 4000 + case, scale=(2.0 / (9 * C)) ** 0.5 * 0.6)
        w[C * 10 + len(dil) * (C * C * 9 + C) + spec.head_channels * C] = 0.2
        frames = rng.integers(80, 3000, size=(n, H, W)).astype(np.uint16)
        ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
        kw = dict(conv_impl=P.CONV_TCGEN05)
        ma = G.gpu_forward_maps(spec, w, frames, ck, fusion=P.FUSE_HEAD, **kw)
        a = G.gpu_localize(spec, w, frames, ck, 0.5, fusion=P.FUSE_HEAD, **kw)
        for fusion in (P.FUSE_AUTO, P.FUSE_PAIRS_1CTA):
            mb = G.gpu_forward_maps(spec, w, frames, ck, fusion=fusion, **kw)
            assert np.array_equal(ma, mb), (case, C, dil, H, W, fusion)
            b = G.gpu_localize(spec, w, frames, ck, 0.5, fusion=fusion, **kw)
            assert len(a) == len(b) and a.tobytes() == b.tobytes(), (case, C, dil, H, W, fusion)
