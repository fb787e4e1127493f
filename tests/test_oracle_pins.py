"""Pins for the CPU oracle (oracle/) against things other than itself.

The paper prints no worked example for the hot path, so the pins are:
  1. brute force on tiny inputs - a SCATTER-form convolution written here in pure Python,
     structurally different from the oracle's gather form;
  2. reduction to a library routine - torch.nn.functional.conv2d in fp64;
  3. hand-derived emitter lists for hand-placed delta maps (tests/golden/delta_maps.json)
     and a rank/maximum_filter formulation of the NMS from scipy;
  4. invariants: zero signal -> bias only, integer-shift equivariance, identity trunk,
     single-tap trunk (pins orientation and dilation), threshold monotonicity,
     non-adjacency, coordinate range; closed forms for the activations and for the
     parameter / FLOP counts of SURVEY.md 8(a).
Each is chosen so that a plausible mistake (dropped term, wrong sign or index, transposed
operand, convolution instead of cross-correlation, wrong padding) fails at least one.
"""
import json
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from smlm_synth import (blob_offsets, blob_size, get_config, he_normal_blob, make_frames,
                        make_weights, NetSpec)

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


# --------------------------------------------------------------------------- helpers
def _tiny_net(C=3, dil=(1, 2), nh=5, stem_relu=1):
    return NetSpec(C, tuple(dil), nh, "fp32", stem_relu=stem_relu)


def _rand_blob(spec, seed, bias=True):
    rng = np.random.default_rng(seed)
    blob = rng.normal(0, 0.4, size=blob_size(spec)).astype(np.float32)
    if not bias:
        off = blob_offsets(spec)
        C, nh = spec.channels, spec.head_channels
        blob[off["stem_b"]:off["stem_b"] + C] = 0
        for l in range(spec.n_layers):
            blob[off[f"b{l}"]:off[f"b{l}"] + C] = 0
        blob[off["head_b"]:off["head_b"] + nh] = 0
    return blob


def _split(spec, blob):
    off = blob_offsets(spec)
    C, nh = spec.channels, spec.head_channels
    IF = spec.in_frames
    out = {"stem_w": blob[off["stem_w"]:off["stem_w"] + C * IF * 9].reshape(C, IF, 3, 3).astype(np.float64),
           "stem_b": blob[off["stem_b"]:off["stem_b"] + C].astype(np.float64), "w": [], "b": []}
    for l in range(spec.n_layers):
        out["w"].append(blob[off[f"w{l}"]:off[f"w{l}"] + C * C * 9].reshape(C, C, 3, 3).astype(np.float64))
        out["b"].append(blob[off[f"b{l}"]:off[f"b{l}"] + C].astype(np.float64))
    out["head_w"] = blob[off["head_w"]:off["head_w"] + nh * C].reshape(nh, C).astype(np.float64)
    out["head_b"] = blob[off["head_b"]:off["head_b"] + nh].astype(np.float64)
    return out


def _scatter_conv(x, w, b, d):
    """Brute force, SCATTER form: every input value is pushed to the outputs it feeds.
    x [Cin][H][W], w [Cout][Cin][3][3]; output pixel (y,x) reads input (y+(ky-1)d, x+(kx-1)d),
    so input pixel (iy,ix) feeds output (iy-(ky-1)d, ix-(kx-1)d)."""
    cin, H, W = x.shape
    cout = w.shape[0]
    out = np.zeros((cout, H, W))
    for co in range(cout):
        out[co] += b[co]
    for ci in range(cin):
        for iy in range(H):
            for ix in range(W):
                v = x[ci, iy, ix]
                for ky in range(3):
                    for kx in range(3):
                        oy, ox = iy - (ky - 1) * d, ix - (kx - 1) * d
                        if 0 <= oy < H and 0 <= ox < W:
                            for co in range(cout):
                                out[co, oy, ox] += w[co, ci, ky, kx] * v
    return out


def _forward_brute(spec, blob, frame, offset, gain):
    p = _split(spec, blob)
    xhat = ((frame.astype(np.float64) - offset) / gain) / spec.norm_scale
    a = _scatter_conv(xhat[None], p["stem_w"], p["stem_b"], 1)
    if spec.stem_relu:
        a = np.maximum(a, 0)
    for l, d in enumerate(spec.dilations):
        a = a + np.maximum(_scatter_conv(a, p["w"][l], p["b"][l], d), 0)
    o = np.einsum("hc,cyx->hyx", p["head_w"], a) + p["head_b"][:, None, None]
    return o, a


def _forward_torch(spec, blob, frames, offset, gain, offset_map=None, gain_map=None):
    import torch
    import torch.nn.functional as F
    p = _split(spec, blob)
    off = torch.from_numpy(np.asarray(offset_map, dtype=np.float64)) if offset_map is not None else offset
    g = torch.from_numpy(np.asarray(gain_map, dtype=np.float64)) if gain_map is not None else gain
    x = ((torch.from_numpy(frames.astype(np.float64)) - off) / g / spec.norm_scale)[:, None]
    a = F.conv2d(x, torch.from_numpy(p["stem_w"]), torch.from_numpy(p["stem_b"]), padding=1)
    if spec.stem_relu:
        a = torch.relu(a)
    layers = [a]
    for l, d in enumerate(spec.dilations):
        t = F.conv2d(a, torch.from_numpy(p["w"][l]), torch.from_numpy(p["b"][l]), padding=d, dilation=d)
        a = a + torch.relu(t)
        layers.append(a)
    o = F.conv2d(a, torch.from_numpy(p["head_w"])[:, :, None, None], torch.from_numpy(p["head_b"]))
    return o.numpy(), [t.numpy() for t in layers]


# --------------------------------------------------------------------------- 1. brute force
@pytest.mark.parametrize("dil", [(1,), (2,), (4,), (1, 2), (2, 4, 1)])
@pytest.mark.parametrize("stem_relu", [0, 1])
def test_forward_matches_bruteforce_scatter(dil, stem_relu):
    spec = _tiny_net(C=3, dil=dil, stem_relu=stem_relu)
    blob = _rand_blob(spec, 11 + len(dil))
    rng = np.random.default_rng(5)
    frame = rng.integers(0, 3000, size=(12, 13)).astype(np.uint16)      # H != W on purpose
    net = O.net_from_spec(spec)
    cam = O.make_camera(100.0, 100.0, 1.7)
    o, dump = O.forward_maps(net, blob, frame[None], cam, dump_trunk=True)
    ob, ab = _forward_brute(spec, blob, frame, 100.0, 1.7)
    assert np.max(np.abs(o[0] - ob)) < 1e-12
    assert np.max(np.abs(dump[0, -1].transpose(2, 0, 1) - ab)) < 1e-12


# --------------------------------------------------------------------------- 2. library routine
def test_forward_matches_torch_conv2d_cfg0():
    cfg = get_config(0)
    fs = make_frames(cfg)
    w = make_weights(cfg)
    net = O.net_from_spec(cfg.net)
    cam = O.make_camera(fs.pixel_size_nm, fs.offset, fs.gain)
    o, dump = O.forward_maps(net, w, fs.frames, cam, dump_trunk=True)
    ot, layers = _forward_torch(cfg.net, w, fs.frames, fs.offset, fs.gain)
    assert np.max(np.abs(o - ot)) < 1e-10
    for l, a in enumerate(layers):
        assert np.max(np.abs(dump[:, l].transpose(0, 3, 1, 2) - a)) < 1e-10, f"layer {l}"


def test_forward_matches_torch_conv2d_cfg1_one_frame():
    cfg = get_config(1)
    fs = make_frames(cfg, 1)
    w = make_weights(cfg, "base")
    w[-cfg.net.head_channels:] = np.linspace(-0.3, 0.4, cfg.net.head_channels)  # non-zero head bias
    net = O.net_from_spec(cfg.net)
    cam = O.make_camera(fs.pixel_size_nm, fs.offset, fs.gain)
    o = O.forward_maps(net, w, fs.frames, cam)
    ot, _ = _forward_torch(cfg.net, w, fs.frames, fs.offset, fs.gain)
    assert np.max(np.abs(o - ot)) < 1e-10


def test_forward_matches_torch_with_camera_maps_and_six_heads():
    spec = NetSpec(8, (1, 2, 4, 8), 6, "fp32")
    blob = _rand_blob(spec, 3)
    rng = np.random.default_rng(9)
    frames = rng.integers(50, 4000, size=(2, 40, 37)).astype(np.uint16)
    offm = rng.normal(100, 2, size=(40, 37)).astype(np.float32)
    gm = np.clip(rng.normal(2.0, 0.1, size=(40, 37)), 0.5, None).astype(np.float32)
    cam = O.make_camera(100.0, 0.0, 1.0, offm, gm)
    o = O.forward_maps(O.net_from_spec(spec), blob, frames, cam)
    ot, _ = _forward_torch(spec, blob, frames, 0.0, 1.0, offm, gm)
    assert np.max(np.abs(o - ot)) < 1e-10


# --------------------------------------------------------------------------- 3. delta maps
def _load_delta_cases():
    with open(os.path.join(GOLDEN, "delta_maps.json"), "r", encoding="utf-8") as fh:
        return json.load(fh)


_DELTA = _load_delta_cases()


@pytest.mark.parametrize("case", _DELTA["cases"], ids=[c["name"] for c in _DELTA["cases"]])
def test_postprocess_hand_placed_delta_maps(case):
    H, W = _DELTA["H"], _DELTA["W"]
    spec = NetSpec(4, (1,), 5, "fp32")
    net = O.net_from_spec(spec)
    cam = O.make_camera(_DELTA["pixel_size_nm"], 100.0, 1.0)
    o = np.zeros((1, 5, H, W))
    o[0, 0] = case["background_logit"]
    for s in case["spikes"]:
        logit = s["logit"] if "logit" in s else math.log(s["p"] / (1.0 - s["p"]))
        o[0, 0, s["y"], s["x"]] = logit
        for h, key in ((1, "o_dx"), (2, "o_dy"), (3, "o_N"), (4, "o_bg")):
            if key in s:
                o[0, h, s["y"], s["x"]] = s[key]
    em = O.postprocess(net, o, cam, case["threshold"])
    exp = sorted(case["expect"], key=lambda e: e["pix"])
    assert [int(p) for p in em["pix"]] == [e["pix"] for e in exp]
    assert all(int(f) == 0 for f in em["frame"])
    for got, e in zip(em, exp):
        for key in ("x_nm", "y_nm", "p", "photons", "bg"):
            if key in e:
                assert got[key] == pytest.approx(e[key], rel=1e-12, abs=1e-30), (case["name"], key)
        assert np.isfinite([got[k] for k in ("x_nm", "y_nm", "z_nm", "photons", "bg", "p")]).all()
        assert got["z_nm"] == 0.0


def test_postprocess_six_heads_z_and_channel_order():
    """n_h = 6 order is (p,dx,dy,z,N,bg) (reading G6): z = 700*tanh(o_z); N reads channel 4."""
    spec = NetSpec(4, (1,), 6, "fp32")
    net = O.net_from_spec(spec)
    cam = O.make_camera(100.0, 100.0, 1.0)
    o = np.zeros((2, 6, 5, 5))
    o[:, 0] = -6.0
    o[1, 0, 2, 2] = 3.0
    o[1, 3, 2, 2] = math.atanh(0.5)        # z -> 350 nm
    o[1, 4, 2, 2] = 40.0                   # N -> 40000
    o[1, 5, 2, 2] = -40.0                  # bg -> ~0
    em = O.postprocess(net, o, cam, 0.3)
    assert len(em) == 1 and em["frame"][0] == 1 and em["pix"][0] == 12
    assert em["z_nm"][0] == pytest.approx(350.0, rel=1e-12)
    assert em["photons"][0] == pytest.approx(40000.0, rel=1e-12)
    assert em["bg"][0] == pytest.approx(100 * 4.248354255291589e-18, rel=1e-9)


def test_postprocess_matches_rank_maximum_filter():
    """NMS with index tie-break == 'the (value, -index) rank equals its 3x3 maximum'
    (scipy.ndimage.maximum_filter with out-of-frame = -1): an independent formulation."""
    from scipy.ndimage import maximum_filter
    rng = np.random.default_rng(42)
    H, W = 37, 41
    spec = NetSpec(4, (1,), 5, "fp32")
    net = O.net_from_spec(spec)
    cam = O.make_camera(100.0, 100.0, 1.0)
    # coarse quantisation => many exact ties
    o = np.zeros((3, 5, H, W))
    o[:, 0] = np.round(rng.normal(0, 1.5, size=(3, H, W)) * 2) / 2
    for thr in (0.0, 0.3, 0.7):
        em = O.postprocess(net, o, cam, thr)
        got = {(int(e["frame"]), int(e["pix"])) for e in em}
        want = set()
        lthr = -np.inf if thr <= 0 else math.log(thr / (1 - thr))
        for f in range(3):
            v = o[f, 0].ravel()
            order = np.lexsort((-np.arange(v.size), v))      # ascending value, then descending index
            rank = np.empty(v.size, dtype=np.int64)
            rank[order] = np.arange(v.size)
            rank = rank.reshape(H, W)
            mx = maximum_filter(rank, size=3, mode="constant", cval=-1)
            for q in np.flatnonzero((rank == mx).ravel() & (v > lthr)):
                want.add((f, int(q)))
        assert got == want
        pts = np.array(sorted(got))
        # non-adjacency inside each frame
        for f in range(3):
            q = pts[pts[:, 0] == f][:, 1]
            yy, xx = q // W, q % W
            dy = np.abs(yy[:, None] - yy[None, :])
            dx = np.abs(xx[:, None] - xx[None, :])
            adj = (np.maximum(dy, dx) == 1)
            assert not adj.any()


# --------------------------------------------------------------------------- 4. invariants
def test_zero_signal_gives_bias_only():
    spec = _tiny_net(C=4, dil=(1, 2, 4))
    cam = O.make_camera(100.0, 100.0, 1.0)
    frames = np.full((1, 40, 40), 100, dtype=np.uint16)       # adu == offset -> xhat == 0
    blob0 = _rand_blob(spec, 1, bias=False)
    blob0[-5:] = [0.1, -0.2, 0.3, -0.4, 0.5]                  # head bias only
    o = O.forward_maps(O.net_from_spec(spec), blob0, frames, cam)
    for h, b in enumerate([0.1, -0.2, 0.3, -0.4, 0.5]):
        assert np.all(o[0, h] == np.float32(b).astype(np.float64))
    blob1 = _rand_blob(spec, 2, bias=True)
    o = O.forward_maps(O.net_from_spec(spec), blob1, frames, cam)
    R = spec.radius
    interior = o[0, :, R:-R, R:-R]
    assert interior.shape[1] > 2
    assert np.max(np.abs(interior - interior[:, :1, :1])) < 1e-13


def test_integer_shift_equivariance():
    cfg = get_config(0)
    spec = cfg.net
    R = spec.radius
    w = make_weights(cfg)
    rng = np.random.default_rng(3)
    H = W = 64
    big = rng.integers(90, 1500, size=(H + 8, W + 8)).astype(np.uint16)
    sy, sx = 3, 5
    f0 = big[0:H, 0:W]
    f1 = big[sy:sy + H, sx:sx + W]                           # content moved by (-sy, -sx)
    cam = O.make_camera(100.0, 100.0, 1.0)
    net = O.net_from_spec(spec)
    o0 = O.forward_maps(net, w, f0[None], cam)[0]
    o1 = O.forward_maps(net, w, f1[None], cam)[0]
    a = o0[:, R + sy:H - R, R + sx:W - R]
    b = o1[:, R:H - R - sy, R:W - R - sx]
    assert a.shape[1] > 10 and np.max(np.abs(a - b)) < 1e-12
    # and it does differ inside the border band (so the test is not vacuous)
    assert np.max(np.abs(o0[:, sy:sy + 4, sx:sx + 4] - o1[:, 0:4, 0:4])) > 1e-6


def test_identity_and_single_tap_trunk():
    spec = _tiny_net(C=3, dil=(2, 4))
    off = blob_offsets(spec)
    rng = np.random.default_rng(8)
    frames = rng.integers(0, 4000, size=(1, 20, 22)).astype(np.uint16)
    cam = O.make_camera(100.0, 100.0, 1.0)
    net = O.net_from_spec(spec)
    blob = _rand_blob(spec, 4, bias=False)
    C = spec.channels
    for l in range(2):
        blob[off[f"w{l}"]:off[f"w{l}"] + C * C * 9] = 0
    _, dump = O.forward_maps(net, blob, frames, cam, dump_trunk=True)
    assert np.array_equal(dump[0, 0], dump[0, 2])            # identity trunk: a_L == a_0
    # single tap (ky, kx) on the diagonal co == ci: a1 = a0 + ReLU(a0 shifted by ((ky-1)d, (kx-1)d))
    for (ky, kx) in [(0, 0), (0, 2), (1, 0), (2, 1), (2, 2)]:
        b2 = blob.copy()
        wl = np.zeros((C, C, 3, 3), dtype=np.float32)
        for c in range(C):
            wl[c, c, ky, kx] = 1.0
        b2[off["w0"]:off["w0"] + C * C * 9] = wl.ravel()
        _, dump = O.forward_maps(net, b2, frames, cam, dump_trunk=True)
        a0, a1 = dump[0, 0], dump[0, 1]
        d = spec.dilations[0]
        H, W = a0.shape[:2]
        shifted = np.zeros_like(a0)
        for y in range(H):
            for x in range(W):
                yy, xx = y + (ky - 1) * d, x + (kx - 1) * d
                if 0 <= yy < H and 0 <= xx < W:
                    shifted[y, x] = a0[yy, xx]
        assert np.max(np.abs(a1 - (a0 + np.maximum(shifted, 0)))) < 1e-14, (ky, kx)


def test_threshold_monotone_nonadjacent_and_coordinate_range():
    cfg = get_config(0)
    fs = make_frames(cfg)
    w = make_weights(cfg)
    net = O.net_from_spec(cfg.net)
    cam = O.make_camera(fs.pixel_size_nm, fs.offset, fs.gain)
    o = O.forward_maps(net, w, fs.frames, cam)
    prev = None
    for thr in (0.0, 0.1, 0.3, 0.5, 0.9, 1.0):
        em = O.postprocess(net, o, cam, thr)
        cur = {(int(e["frame"]), int(e["pix"])) for e in em}
        if prev is not None:
            assert cur <= prev
        prev = cur
        W = fs.frames.shape[2]
        ix, iy = em["pix"] % W, em["pix"] // W
        assert np.all(np.abs(em["x_nm"] / 100.0 - ix) < 0.5) and np.all(np.abs(em["y_nm"] / 100.0 - iy) < 0.5)
        key = em["frame"].astype(np.int64) * (1 << 32) + em["pix"]
        assert np.all(np.diff(key) > 0)                       # O8: sorted by (frame, pix), unique
    assert len(prev) == 0
    em = O.postprocess(net, o, cam, 0.3)
    assert len(em) > 50                                        # cfg 0 literal weights do detect


def test_activation_closed_forms():
    spec = NetSpec(4, (1,), 6, "fp32")
    net = O.net_from_spec(spec)
    v = np.array([-40.0, -1.0, 0.0, math.atanh(0.5), 1.0, 40.0])
    o = np.zeros((1, 6, 1, v.size))
    o[0, :, 0, :] = v
    act = O.activate_maps(net, o)[0, :, 0, :]
    assert act[0, 2] == 0.5 and act[0, 4] == pytest.approx(1 / (1 + math.exp(-1)), rel=1e-15)
    assert act[0, 1] == pytest.approx(1 - 1 / (1 + math.exp(-1)), rel=1e-14)
    assert act[1, 3] == pytest.approx(0.25, rel=1e-15) and act[2, 5] == 0.5 and act[2, 0] == -0.5
    assert act[3, 3] == pytest.approx(0.5, rel=1e-15)          # z map is plain tanh
    assert act[4, 2] == pytest.approx(math.log(2.0), rel=1e-15)
    assert act[5, 4] == pytest.approx(math.log1p(math.e), rel=1e-15)
    assert act[4, 5] == pytest.approx(40.0, rel=1e-15) and act[4, 0] == pytest.approx(math.exp(-40), rel=1e-12)
    assert np.isfinite(act).all()


def test_closed_form_counts():
    want = {0: (9525, 18880, 16), 1: (250133, 499008, 46), 2: (444166, 886656, 46),
            3: (250133, 499008, 46), 4: (250133, 499008, 46)}
    for i, (params, flop, radius) in want.items():
        spec = get_config(i).net
        assert spec.n_params() == params and spec.flop_per_px() == flop and spec.radius == radius
        assert he_normal_blob(spec, 1).size == params
        assert O.lib().smlm_oracle_blob_size(O.net_from_spec(spec)) == params


def test_halo_46_is_exact_and_45_is_not():
    """Tiling reading G15: the maps of a crop equal the whole-frame maps exactly R = 46 px
    inside the crop, and not at 45 (so the receptive-field radius is pinned)."""
    cfg = get_config(1)
    spec = cfg.net
    w = make_weights(cfg, "base")
    fs = make_frames(cfg, 1, height=140, width=140)
    net = O.net_from_spec(spec)
    cam = O.make_camera(100.0, fs.offset, fs.gain)
    whole = O.forward_maps(net, w, fs.frames, cam)[0]
    crop = O.forward_maps(net, w, fs.frames[:, :120, :120], cam)[0]
    R = spec.radius
    assert np.max(np.abs(whole[:, :120 - R, :120 - R] - crop[:, :120 - R, :120 - R])) == 0.0
    assert np.max(np.abs(whole[:, :120 - R + 1, :120 - R + 1] - crop[:, :120 - R + 1, :120 - R + 1])) > 0.0


# --------------------------------------------------------------------------- 3-frame temporal context (G24)
def _context_stack(frames):
    """[n][H][W] -> [n][3][H][W]: frames f-1, f, f+1 with indices clamped to the call."""
    n = len(frames)
    idx = np.clip(np.arange(n)[:, None] + np.array([-1, 0, 1])[None], 0, n - 1)
    return frames[idx]


def test_three_frame_stem_matches_torch_conv2d():
    """in_frames = 3: the stem is a 3 -> C convolution over the
    normalised frames f-1, f, f+1 (clamped).  Library routine: torch conv2d in fp64 on the
    explicitly built 3-channel input; catches a wrong channel order, a wrong clamp and a
    wrong weight stride."""
    import torch
    import torch.nn.functional as F
    spec = NetSpec(6, (1, 2), 5, "fp32", in_frames=3)
    blob = _rand_blob(spec, 21)
    rng = np.random.default_rng(4)
    frames = rng.integers(50, 4000, size=(5, 17, 19)).astype(np.uint16)
    net = O.net_from_spec(spec)
    cam = O.make_camera(100.0, 90.0, 1.3)
    o, dump = O.forward_maps(net, blob, frames, cam, dump_trunk=True)
    p = _split(spec, blob)
    x = torch.from_numpy(((_context_stack(frames).astype(np.float64) - 90.0) / 1.3) / spec.norm_scale)
    a = torch.relu(F.conv2d(x, torch.from_numpy(p["stem_w"]), torch.from_numpy(p["stem_b"]), padding=1))
    assert np.max(np.abs(dump[:, 0].transpose(0, 3, 1, 2) - a.numpy())) < 1e-12
    for l, d in enumerate(spec.dilations):
        a = a + torch.relu(F.conv2d(a, torch.from_numpy(p["w"][l]), torch.from_numpy(p["b"][l]), padding=d, dilation=d))
    ot = F.conv2d(a, torch.from_numpy(p["head_w"])[:, :, None, None], torch.from_numpy(p["head_b"])).numpy()
    assert np.max(np.abs(o - ot)) < 1e-10


def test_three_frame_stem_reduces_to_single_frame_and_pins_channel_order():
    """Weights on the centre channel only == the 1-frame network on the same frames; weights
    on channel 0 (or 2) only == the 1-frame network on the sequence shifted by one frame with
    the first (last) frame repeated: pins which channel is f-1 and the clamp at both ends."""
    spec1 = NetSpec(4, (1, 2), 5, "fp32")
    spec3 = NetSpec(4, (1, 2), 5, "fp32", in_frames=3)
    b1 = _rand_blob(spec1, 33)
    rng = np.random.default_rng(6)
    frames = rng.integers(50, 4000, size=(4, 11, 12)).astype(np.uint16)
    cam = O.make_camera(100.0, 100.0, 1.0)
    o1 = O.forward_maps(O.net_from_spec(spec1), b1, frames, cam)
    C = spec1.channels
    for ch, seq in ((1, frames), (0, frames[[0, 0, 1, 2]]), (2, frames[[1, 2, 3, 3]])):
        w3 = np.zeros((C, 3, 3, 3), dtype=np.float32)
        w3[:, ch] = b1[:C * 9].reshape(C, 3, 3)
        b3 = np.concatenate([w3.ravel(), b1[C * 9:]])
        assert b3.size == blob_size(spec3)
        o3 = O.forward_maps(O.net_from_spec(spec3), b3, frames, cam)
        ref = o1 if ch == 1 else O.forward_maps(O.net_from_spec(spec1), b1, seq, cam)
        assert np.array_equal(o3, ref), f"channel {ch}"


def test_three_frame_stem_bruteforce_scatter():
    spec = NetSpec(3, (2,), 5, "fp32", in_frames=3)
    blob = _rand_blob(spec, 8)
    rng = np.random.default_rng(2)
    frames = rng.integers(0, 3000, size=(3, 9, 10)).astype(np.uint16)
    o, dump = O.forward_maps(O.net_from_spec(spec), blob, frames, O.make_camera(100.0, 100.0, 1.7), dump_trunk=True)
    p = _split(spec, blob)
    ctx = _context_stack(frames)
    for f in range(3):
        xhat = ((ctx[f].astype(np.float64) - 100.0) / 1.7) / spec.norm_scale
        a = np.maximum(_scatter_conv(xhat, p["stem_w"], p["stem_b"], 1), 0)
        assert np.max(np.abs(dump[f, 0].transpose(2, 0, 1) - a)) < 1e-12
