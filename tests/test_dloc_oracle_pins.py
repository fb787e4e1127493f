"""Pins of oracle/dloc_oracle.c (the paper's DilatedLoc topology; P:57-61,
P:144), CPU only.  Nothing here comes from the CUDA path.

The paper prints no worked example of this network (no widths, Figure 2 is a picture), so
numerical parity WITH THE PAPER is unpinned; the oracle is pinned to mathematics instead:
  * every stage against torch.nn.functional in fp64 (conv2d with dilation / padding,
    max_pool2d, interpolate(nearest), concatenation order) - an independent library;
  * brute-force scatter-form convolution over a concatenated input (dense connection:
    channel order, dilation sign, zero padding);
  * hand-computed tiny cases: pooling of an odd-sized map, up-sampling index rule,
    uncertainty decode at 0 and +-40;
  * invariants: zero signal -> maps that depend on biases only; the 3-frame input clamps at
    the ends of the stack; parameter count = closed form.
"""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import dloc as D
from oracle import oracle as O
from smlm_synth import DlocSpec, dloc_he_normal_blob


def _split(spec, blob):
    out, p = {}, 0
    for name, co, ci, k in spec.layers():
        w = blob[p:p + co * ci * k * k].reshape(co, ci, k, k)
        p += w.size
        out[name] = (torch.from_numpy(w.astype(np.float64)), torch.from_numpy(blob[p:p + co].astype(np.float64)))
        p += co
    assert p == blob.size
    return out


def _torch_forward(spec, blob, frames, offset=100.0, gain=1.0):
    """The same network written with torch.nn.functional ops in fp64 (independent code)."""
    P = _split(spec, blob)
    n, H, W = frames.shape
    x = (torch.from_numpy(frames.astype(np.float64)) - offset) / gain / spec.norm_scale
    if spec.in_frames == 3:
        idx = [np.clip(np.arange(n) + s, 0, n - 1) for s in (-1, 0, 1)]
        x = torch.stack([x[i] for i in idx], dim=1)
    else:
        x = x[:, None]
    dump = {}
    w, b = P["stem"]
    f = F.conv2d(x, w, b, padding=1)
    f = F.relu(f) if spec.stem_relu else f
    dump["stem"] = f
    for blk in range(spec.n_blocks):
        feats = [f]
        for i, d in enumerate(spec.dilations):
            w, b = P[f"b{blk}l{i}"]
            feats.append(F.relu(F.conv2d(torch.cat(feats, 1), w, b, padding=d, dilation=d)))
        w, b = P[f"b{blk}t"]
        f = F.relu(F.conv2d(torch.cat(feats, 1), w, b))
        dump[f"block{blk}"] = f
    e0 = f
    e1 = F.relu(F.conv2d(F.max_pool2d(e0, 2), *P["enc1"], padding=1))
    e2 = F.relu(F.conv2d(F.max_pool2d(e1, 2), *P["enc2"], padding=1))
    def up(t, size):
        # library routines only: nearest x 2, then the finer map's odd last row / column (if any)
        # by replicating the edge (reading D5)
        u = F.interpolate(t, scale_factor=2, mode="nearest")
        return F.pad(u, (0, size[1] - u.shape[3], 0, size[0] - u.shape[2]), mode="replicate")
    m1 = F.relu(F.conv2d(torch.cat([up(e2, e1.shape[2:]), e1], 1), *P["dec1"], padding=1))
    m0 = F.relu(F.conv2d(torch.cat([up(m1, e0.shape[2:]), e0], 1), *P["dec0"], padding=1))
    dump.update(e1=e1, e2=e2, m1=m1, m0=m0)
    o = F.conv2d(m0, *P["head"])
    return o.numpy(), {k: v.numpy() for k, v in dump.items()}


@pytest.mark.parametrize("c0,g,nb,dil,inf,H,W,relu", [(8, 4, 2, (1, 2), 1, 12, 16, 1), (16, 8, 4, (2, 4, 8, 16), 1, 40, 36, 1),
                                                       (8, 8, 1, (2, 4), 3, 13, 11, 0), (12, 4, 3, (1, 3, 2), 3, 9, 22, 1)])
def test_every_stage_equals_torch_functional_fp64(c0, g, nb, dil, inf, H, W, relu):
    spec = DlocSpec(c0=c0, growth=g, n_blocks=nb, dilations=dil, in_frames=inf, stem_relu=relu)
    blob = dloc_he_normal_blob(spec, 3)
    blob += np.random.default_rng(1).normal(0, 0.05, blob.size).astype(np.float32)        # non-zero biases too
    frames = np.random.default_rng(H).integers(90, 3000, size=(4, H, W)).astype(np.uint16)
    net = D.net_from_spec(spec)
    assert D.blob_size(net) == spec.n_params() == blob.size
    o, dump = D.forward_maps(net, blob, frames, O.make_camera(100.0, 100.0, 1.0), dump=True)
    ot, dt = _torch_forward(spec, blob, frames)
    for f in range(4):
        for name, _ in D.dump_shapes(net, H, W):
            scale = max(1.0, float(np.abs(dt[name][f]).max()))
            assert np.max(np.abs(dump[f][name] - dt[name][f])) < 1e-10 * scale, (f, name)
    assert np.max(np.abs(o - ot)) < 1e-9 * max(1.0, float(np.abs(ot).max()))


def test_dense_connection_by_brute_force_scatter():
    """One DCD layer on a concatenated input, scatter form (each input value is added to the
    outputs it reaches): pins channel order of the concatenation, dilation sign, padding."""
    spec = DlocSpec(c0=3, growth=2, n_blocks=1, dilations=(2, 3), in_frames=1)
    rng = np.random.default_rng(7)
    blob = rng.normal(0, 0.4, spec.n_params()).astype(np.float32)
    H, W = 9, 10
    frames = rng.integers(100, 2000, size=(1, H, W)).astype(np.uint16)
    net = D.net_from_spec(spec)
    _, dump = D.forward_maps(net, blob, frames, O.make_camera(100.0, 100.0, 1.0), dump=True)
    P = _split(spec, blob)
    f0 = dump[0]["stem"]
    g = [f0]
    for i, d in enumerate(spec.dilations):
        x = np.concatenate(g, 0)
        w, b = (t.numpy() for t in P[f"b0l{i}"])
        out = np.tile(b[:, None, None], (1, H, W)).astype(np.float64)
        for ci in range(x.shape[0]):
            for y in range(H):
                for xx in range(W):
                    for ky in range(3):
                        for kx in range(3):
                            yo, xo = y - (ky - 1) * d, xx - (kx - 1) * d          # output reached by tap (ky,kx)
                            if 0 <= yo < H and 0 <= xo < W:
                                out[:, yo, xo] += w[:, ci, ky, kx] * x[ci, y, xx]
        g.append(np.maximum(out, 0))
    w, b = (t.numpy() for t in P["b0t"])
    t = np.maximum(np.einsum("oc,chw->ohw", w[:, :, 0, 0], np.concatenate(g, 0)) + b[:, None, None], 0)
    assert np.max(np.abs(t - dump[0]["block0"])) < 1e-10


def test_upsample2_against_interpolate_and_by_hand():
    """Reading D5 ("two-stage U-Net"; P:192 item 2): nearest neighbour x 2 to exactly the finer
    map's size.  Even sizes: torch's nearest interpolation.  Odd target: written out by hand."""
    import torch
    import torch.nn.functional as F
    rng = np.random.default_rng(3)
    for c, H, W in ((1, 1, 1), (3, 4, 6), (2, 5, 3)):
        x = rng.normal(size=(c, H, W))
        ref = F.interpolate(torch.from_numpy(x)[None], scale_factor=2, mode="nearest")[0].numpy()
        assert np.array_equal(D.upsample2(x, 2 * H, 2 * W), ref)
    x = np.array([[[1., 2., 3.], [4., 5., 6.], [7., 8., 9.]]])
    want = np.array([[1, 1, 2, 2, 3, 3, 3],
                     [1, 1, 2, 2, 3, 3, 3],
                     [4, 4, 5, 5, 6, 6, 6],
                     [4, 4, 5, 5, 6, 6, 6],
                     [7, 7, 8, 8, 9, 9, 9],
                     [7, 7, 8, 8, 9, 9, 9],
                     [7, 7, 8, 8, 9, 9, 9]], dtype=np.float64)
    assert np.array_equal(D.upsample2(x, 7, 7)[0], want)
    assert np.array_equal(D.upsample2(x, 6, 7)[0], want[:6]) and np.array_equal(D.upsample2(x, 7, 6)[0], want[:, :6])
    two = np.stack([x[0], -x[0].T])                       # channels stay apart, rows are not columns
    got = D.upsample2(two, 7, 7)
    assert np.array_equal(got[0], want) and np.array_equal(got[1], -want.T)


def test_maxpool2_against_max_pool2d_and_by_hand_on_an_odd_map():
    """Reading D4: 2 x 2 max pooling, stride 2, floor - the trailing odd row / column is dropped."""
    import torch
    import torch.nn.functional as F
    rng = np.random.default_rng(4)
    for c, H, W in ((1, 2, 2), (3, 6, 8), (2, 7, 5), (2, 4, 9)):
        x = rng.normal(size=(c, H, W))
        assert np.array_equal(D.maxpool2(x), F.max_pool2d(torch.from_numpy(x)[None], 2)[0].numpy())
    x = np.array([[[1, 9, 2, 3, 50],
                   [4, 5, 8, 7, 51],
                   [-1, -2, -3, -4, 52],
                   [-8, -7, -6, -5, 53],
                   [60, 61, 62, 63, 64]]], dtype=np.float64)
    assert np.array_equal(D.maxpool2(x)[0], np.array([[9., 8.], [-1., -3.]]))   # row 4 / column 4 never read


def test_uncertainty_decode_by_hand():
    spec = DlocSpec(c0=8, growth=4)
    o = np.zeros((1, 10, 4, 4))
    o[0, 0] = -5.0
    o[0, 0, 1, 2] = 5.0
    o[0, 6, 1, 2], o[0, 7, 1, 2], o[0, 8, 1, 2], o[0, 9, 1, 2] = 0.0, 40.0, -40.0, np.log(3.0)
    em = D.postprocess(spec, o, O.make_camera(100.0, 100.0, 1.0), 0.3)
    assert len(em) == 1 and em["pix"][0] == 6
    assert em["sx_nm"][0] == pytest.approx(3.0 * 0.5 * 100.0)          # sigma_xy_px * sigmoid(0) * pixel
    assert em["sy_nm"][0] == pytest.approx(300.0) and em["sz_nm"][0] == pytest.approx(0.0, abs=1e-12)
    assert em["s_photons"][0] == pytest.approx(1000.0 * 0.75)          # sigmoid(ln 3) = 3/4
    assert em["z_nm"][0] == 0.0 and em["x_nm"][0] == pytest.approx(200.0)


def test_zero_signal_gives_bias_only_maps_and_context_clamps():
    spec = DlocSpec(c0=8, growth=4, n_blocks=2, dilations=(2, 4), in_frames=3)
    blob = dloc_he_normal_blob(spec, 5)
    net = D.net_from_spec(spec)
    cam = O.make_camera(100.0, 100.0, 1.0)
    z = np.full((3, 12, 12), 100, np.uint16)                     # adu == offset: xhat == 0, biases zero
    assert np.max(np.abs(D.forward_maps(net, blob, z, cam))) == 0.0
    rng = np.random.default_rng(0)
    fr = rng.integers(100, 2000, size=(3, 12, 12)).astype(np.uint16)
    o = D.forward_maps(net, blob, fr, cam)
    # frame 0 sees (0, 0, 1): the same as a stack (0, 0, 1) evaluated at its middle frame
    o2 = D.forward_maps(net, blob, fr[[0, 0, 1]], cam)
    assert np.array_equal(o[0], o2[1])
    o3 = D.forward_maps(net, blob, fr[[1, 2, 2]], cam)
    assert np.array_equal(o[2], o3[1])
    assert DlocSpec().n_params() == D.blob_size(D.net_from_spec(DlocSpec()))
