"""GPU parity tests of the paper's own topology (include/dloc.h) against
oracle/dloc_oracle.c on the same seeded inputs: every dumped feature map and the ten head maps
element by element, the emitter list through the parity gate, the uncertainties at matched
detections.  fp32 reference mode at 1e-4; bf16 (tcgen05 and the CUDA-core twin) at 2e-2."""
import dataclasses

import numpy as np
import pytest

from oracle import dloc as D
from oracle import oracle as O
from smlm_synth import DlocSpec, dloc_he_normal_blob
import paper_2410_02314_b200 as P
import gpu_util as G

pytestmark = pytest.mark.gpu


def _frames(n, H, W, seed):
    rng = np.random.default_rng(seed)
    base = rng.integers(90, 400, size=(n, H, W)).astype(np.float64)
    yy, xx = np.mgrid[0:H, 0:W]
    for f in range(n):                       # a few Gaussian blobs so that the p-map has structure
        for _ in range(max(4, H * W // 600)):
            cy, cx, a = rng.uniform(0, H), rng.uniform(0, W), rng.uniform(500, 4000)
            base[f] += a * np.exp(-((yy - cy) ** 2 + (xx - cx) ** 2) / (2 * 1.3 ** 2))
    return np.clip(base, 0, 65535).astype(np.uint16)


def _gpu_maps(spec, w, frames, ck, dump=False, **kw):
    torch = G.torch_mod()
    n, H, W = frames.shape
    with P.DlocLocalizer(P.dloc_desc_from_spec(spec, **kw), w) as loc:
        fr = torch.from_numpy(frames).cuda()
        maps = torch.empty((n, P.DLOC_HEADS, H, W), dtype=torch.float32, device="cuda")
        shapes = D.dump_shapes(D.net_from_spec(spec), H, W)
        per = sum(int(np.prod(s)) for _, s in shapes)
        dbuf = torch.empty((n, per), dtype=torch.float32, device="cuda") if dump else None
        loc.forward_maps(fr, loc.camera(**ck), maps, dbuf)
        torch.cuda.synchronize()
        assert loc.check() == P.OK, loc.last_error()
        o = maps.cpu().numpy()
        if not dump:
            return o
        d = dbuf.cpu().numpy()
        out = []
        for f in range(n):
            m, off = {}, 0
            for name, s in shapes:
                k = int(np.prod(s))
                m[name] = d[f, off:off + k].reshape(s)
                off += k
            out.append(m)
        return o, out


def _gpu_localize(spec, w, frames, ck, thr, host_frames=False, host_out=False, capacity=None, **kw):
    torch = G.torch_mod()
    n, H, W = frames.shape
    cap = n * ((H + 1) // 2) * ((W + 1) // 2) if capacity is None else capacity
    with P.DlocLocalizer(P.dloc_desc_from_spec(spec, **kw), w) as loc:
        fr = torch.from_numpy(frames)
        fr = fr.pin_memory() if host_frames else fr.cuda()
        buf = torch.zeros(max(cap, 1) * 48, dtype=torch.uint8)
        buf = buf.pin_memory() if host_out else buf.cuda()
        cnt = loc.localize(fr, loc.camera(**ck), thr, buf, cap)
        torch.cuda.synchronize()
        status = loc.check()
        found = int(cnt.value)
        em = P.dloc_emitters_to_numpy(buf, min(found, cap))
        launches = loc.launch_count()
    return em, found, status, launches


def _spec_for_gate(spec):
    """NetSpec-like view (six-head decode) for gpu_util.parity_gate / activated."""
    import types
    return types.SimpleNamespace(head_channels=6, xy_scale=spec.xy_scale, z_scale_nm=spec.z_scale_nm)


CASES = [pytest.param(DlocSpec(c0=16, growth=16, n_blocks=2, dilations=(1, 2)), 3, 20, 28, id="small"),
         pytest.param(DlocSpec(c0=32, growth=16, n_blocks=2, dilations=(2, 4, 8, 16)), 2, 37, 150, id="ragged-d16"),
         pytest.param(DlocSpec(), 2, 64, 140, id="paper-default")]


@pytest.mark.parametrize("spec,n,H,W", CASES)
def test_dloc_fp32_reference_mode_every_feature_map(spec, n, H, W):
    w = dloc_he_normal_blob(spec, 3, head_gain=0.5)
    frames = _frames(n, H, W, 17)
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    cam = O.make_camera(**ck)
    o, dump = D.forward_maps(D.net_from_spec(spec), w, frames, cam, dump=True)
    og, dg = _gpu_maps(spec, w, frames, ck, dump=True)
    for f in range(n):
        for name in dump[f]:
            sc = max(1.0, float(np.max(np.abs(dump[f][name]))))
            err = float(np.max(np.abs(dg[f][name] - dump[f][name])))
            assert err < 2e-5 * sc, (f, name, err, sc)
    assert np.max(np.abs(og - o)) < 1e-4 * max(1.0, float(np.max(np.abs(o))))
    a_o, a_g = G.activated(_spec_for_gate(spec), o[:, :6]), G.activated(_spec_for_gate(spec), og[:, :6])
    assert np.max(np.abs(a_o - a_g)) < 1e-4
    sig = lambda v: 1.0 / (1.0 + np.exp(-v))
    assert np.max(np.abs(sig(o[:, 6:]) - sig(og[:, 6:].astype(np.float64)))) < 1e-4


@pytest.mark.parametrize("impl", [pytest.param(P.CONV_DIRECT, id="direct"), pytest.param(P.CONV_TCGEN05, id="tcgen05"),
                                  pytest.param(P.CONV_AUTO, id="auto")])
@pytest.mark.parametrize("spec,n,H,W", CASES)
def test_dloc_bf16_maps_and_emitters(spec, n, H, W, impl):
    spec = dataclasses.replace(spec, precision="bf16")
    w = dloc_he_normal_blob(spec, 3, head_gain=0.5)
    frames = _frames(n, H, W, 17)
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    cam = O.make_camera(**ck)
    o, dump = D.forward_maps(D.net_from_spec(spec), w, frames, cam, dump=True)
    og, dg = _gpu_maps(spec, w, frames, ck, dump=True, conv_impl=impl)
    rel = {}
    for name in dump[0]:
        sc = max(1.0, float(max(np.max(np.abs(dump[f][name])) for f in range(n))))
        rel[name] = float(max(np.max(np.abs(dg[f][name] - dump[f][name])) for f in range(n))) / sc
        assert rel[name] < 3e-2, (name, rel[name])
    gs = _spec_for_gate(spec)
    err = G.head_errors(gs, o[:, :6], og[:, :6])
    sig = lambda v: 1.0 / (1.0 + np.exp(-np.asarray(v, dtype=np.float64)))
    err_s = float(np.max(np.abs(sig(o[:, 6:]) - sig(og[:, 6:]))))
    assert err.max() < 2e-2 and err_s < 2e-2, (err, err_s)
    thr = 0.5
    em_o = D.postprocess(spec, o, cam, thr)
    em_g, found, status, launches = _gpu_localize(spec, w, frames, ck, thr, conv_impl=impl)
    assert status == P.OK and found == len(em_g)
    st = G.parity_gate(gs, o[:, :6], em_o, em_g, thr, 2e-2, 100.0, H, W, dp_measured=G.p_error(o, og), o_gpu=og)
    # uncertainties at matched detections: within 2e-2 of their scale
    go = {(int(e["frame"]), int(e["pix"])): e for e in em_o}
    ds = 0.0
    for e in em_g:
        k = (int(e["frame"]), int(e["pix"]))
        if k in go:
            a = go[k]
            ds = max(ds, abs(a["sx_nm"] - e["sx_nm"]) / (spec.sigma_xy_px * 100.0),
                     abs(a["sy_nm"] - e["sy_nm"]) / (spec.sigma_xy_px * 100.0),
                     abs(a["sz_nm"] - e["sz_nm"]) / spec.sigma_z_nm,
                     abs(a["s_photons"] - e["s_photons"]) / spec.sigma_photons)
    assert ds < 2e-2, ds
    name = {P.CONV_DIRECT: "direct", P.CONV_TCGEN05: "tcgen05", P.CONV_AUTO: "auto"}[impl]
    G.record(f"dloc_bf16_{name}_c{spec.c0}g{spec.growth}_{H}x{W}", gate=st, head_max_err=err, sigma_head_err=err_s,
             feature_rel_err=rel, sigma_rel_err=ds, launches=launches)


def test_dloc_tcgen05_matches_direct_bf16_feature_maps():
    """Same rounding points in both 16-bit kernels (bf16 maps and weights, fp32 accumulate, one
    RNE store): only the summation order differs."""
    spec = DlocSpec(c0=32, growth=16, n_blocks=2, dilations=(2, 4, 8, 16), precision="bf16")
    w = dloc_he_normal_blob(spec, 5, head_gain=0.5)
    frames = _frames(2, 45, 200, 3)
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    oa, da = _gpu_maps(spec, w, frames, ck, dump=True, conv_impl=P.CONV_DIRECT)
    for impl in (P.CONV_TCGEN05, P.CONV_AUTO):     # generic tcgen05 kernel / dense-block layers through conv_chain.cu
        ob, db = _gpu_maps(spec, w, frames, ck, dump=True, conv_impl=impl)
        for f in range(2):
            assert np.array_equal(da[f]["stem"], db[f]["stem"])
            for name in da[f]:
                d = np.abs(da[f][name] - db[f][name]) / np.maximum(np.abs(da[f][name]), 1.0)
                assert d.max() < 2.0 ** -5 and np.mean(d > 0) < 0.5, (impl, name, d.max(), np.mean(d > 0))   # bf16 ulps pile up with depth


def test_dloc_pipeline_host_ring_micro_batches_three_frames_and_edges():
    spec = DlocSpec(c0=16, growth=16, n_blocks=2, dilations=(2, 4), in_frames=3, precision="bf16")
    w = dloc_he_normal_blob(spec, 9, head_gain=0.5)
    frames = _frames(7, 24, 40, 21)
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    cam = O.make_camera(**ck)
    o = D.forward_maps(D.net_from_spec(spec), w, frames, cam)
    og = _gpu_maps(spec, w, frames, ck)
    assert G.head_errors(_spec_for_gate(spec), o[:, :6], og[:, :6]).max() < 2e-2
    ref, found, status, _ = _gpu_localize(spec, w, frames, ck, 0.5)
    assert status == P.OK and found == len(ref) and found > 10
    for kw in (dict(micro_batch=2), dict(host_frames=True, micro_batch=2), dict(host_frames=True, host_out=True, micro_batch=3),
               dict(host_out=True)):
        em, f2, st2, _ = _gpu_localize(spec, w, frames, ck, 0.5, **kw)
        assert st2 == P.OK and np.array_equal(em, ref), kw
    # overflow: counted, first `capacity` records kept, reported by dloc_check
    em, f3, st3, _ = _gpu_localize(spec, w, frames, ck, 0.5, capacity=3)
    assert f3 == found and len(em) == 3 and st3 == P.ERR_OVERFLOW
    # empty input, threshold 1 (nothing), threshold 0 (every local maximum)
    em, f4, st4, _ = _gpu_localize(spec, w, frames[:0], ck, 0.5, capacity=4)
    assert f4 == 0 and st4 == P.OK
    em, f5, st5, _ = _gpu_localize(spec, w, frames, ck, 1.0)
    assert f5 == 0 and st5 == P.OK
    em, f6, st6, _ = _gpu_localize(spec, w, frames, ck, 0.0)
    assert st6 == P.OK and f6 >= found
    # bad descriptors are refused
    for kw in (dict(c0=24), dict(growth=8), dict(dilations=(17,)), dict(in_frames=2), dict(n_blocks=0)):
        with pytest.raises(P.SmlmError) as ei:
            P.DlocLocalizer(P.dloc_desc_from_spec(spec, **kw), w)
        assert ei.value.status == P.ERR_INVALID_ARG


def test_dloc_full_size_in_bench_launch_shape_sampled_against_oracle():
    """The shape bench.py --net dloc times: the default DilatedLoc spec in bf16 on 256 x 256 frames,
    default launch sets (64 frames: one full set + a tail), pinned host frames in, pinned host
    list out.  The stack cycles 2 distinct frames, so (1) frames 0 and 65 - one in each launch
    set - are compared element by element with the oracle (head maps through the activations,
    2e-2), (2) every frame's map and emitter records must equal, bit by bit, those of the first
    occurrence of the same distinct frame (position in a launch set must not matter: the chain
    kernel's lane ranges start and end mid-chain), (3) frame 0's emitters go through the gate."""
    spec = DlocSpec(precision="bf16")
    w = dloc_he_normal_blob(spec, 3, head_gain=0.5)
    base = _frames(2, 256, 256, 31)
    n = 66
    frames = np.ascontiguousarray(np.concatenate([base] * (n // 2)))
    ck = dict(pixel_size_nm=100.0, offset=100.0, gain=1.0)
    cam = O.make_camera(**ck)
    o = D.forward_maps(D.net_from_spec(spec), w, base, cam)
    og = _gpu_maps(spec, w, frames, ck)
    for f in range(2, n):
        assert np.array_equal(og[f], og[f % 2]), f
    gs = _spec_for_gate(spec)
    for f in (0, 65):
        err = G.head_errors(gs, o[f % 2:f % 2 + 1, :6], og[f:f + 1, :6])
        assert err.max() < 2e-2, (f, err)
    thr = 0.5
    em, found, status, _ = _gpu_localize(spec, w, frames, ck, thr, host_frames=True, host_out=True)
    assert status == P.OK and found == len(em) and found > 100
    key = lambda e: (int(e["pix"]), float(e["x_nm"]), float(e["y_nm"]), float(e["p"]), float(e["sx_nm"]))
    per = {}
    for e in em:
        per.setdefault(int(e["frame"]), []).append(key(e))
    for f in range(2, n):
        assert sorted(per.get(f, [])) == sorted(per.get(f % 2, [])), f
    em_o = D.postprocess(spec, o[:1], cam, thr)
    em0 = em[em["frame"] == 0]
    st = G.parity_gate(gs, o[:1, :6], em_o, em0, thr, 2e-2, 100.0, 256, 256, dp_measured=G.p_error(o[:1], og[:1]), o_gpu=og[:1])
    G.record("dloc_full_size_256", gate=st, frames=n, emitters=int(found))
