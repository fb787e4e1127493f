"""Helpers shared by the GPU parity tests: run the CUDA library through its C ABI binding,
run the oracle on the same seeded inputs, and apply the parity gate of DESIGN.md."""
from __future__ import annotations

import numpy as np

from oracle import oracle as O
import paper_2410_02314_b200 as P


def torch_mod():
    import torch
    return torch


def gpu_forward_maps(spec, weights, frames, cam_kw, dump_trunk=False, **desc_kw):
    """-> o [n][n_h][H][W] float32 (pre-activation) [, trunk [n][L+1][H][W][C]]"""
    torch = torch_mod()
    desc = P.desc_from_spec(spec, **desc_kw)
    n, H, W = frames.shape
    with P.Localizer(desc, weights) as loc:
        fr = torch.from_numpy(np.ascontiguousarray(frames)).cuda()
        keep = []
        kw = dict(cam_kw)
        for k in ("offset_map", "gain_map"):
            if kw.get(k) is not None:
                t = torch.from_numpy(np.ascontiguousarray(kw[k], dtype=np.float32)).cuda()
                keep.append(t)
                kw[k] = t
        cam = loc.camera(**kw)
        maps = torch.empty((n, spec.head_channels, H, W), dtype=torch.float32, device="cuda")
        trunk = None
        if dump_trunk:
            trunk = torch.empty((n, spec.n_layers + 1, H, W, spec.channels), dtype=torch.float32,
                                device="cuda")
        loc.forward_maps(fr, cam, maps, trunk)
        torch.cuda.synchronize()
        assert loc.check() == P.OK, loc.last_error()
        out = maps.cpu().numpy()
        tr = trunk.cpu().numpy() if dump_trunk else None
    return (out, tr) if dump_trunk else out


def gpu_localize(spec, weights, frames, cam_kw, threshold, capacity=None, host_frames=False,
                 host_out=False, return_status=False, **desc_kw):
    """The whole hot path through smlm_localize -> structured array sorted by (frame, pix)."""
    torch = torch_mod()
    desc = P.desc_from_spec(spec, **desc_kw)
    n, H, W = frames.shape
    if capacity is None:
        capacity = max(1, n * ((H + 1) // 2) * ((W + 1) // 2))
    with P.Localizer(desc, weights) as loc:
        fr = torch.from_numpy(np.ascontiguousarray(frames))
        fr = fr.pin_memory() if host_frames else fr.cuda()
        kw = dict(cam_kw)
        keep = []
        for k in ("offset_map", "gain_map"):
            if kw.get(k) is not None:
                t = torch.from_numpy(np.ascontiguousarray(kw[k], dtype=np.float32)).cuda()
                keep.append(t)
                kw[k] = t
        cam = loc.camera(**kw)
        if host_out:
            buf = torch.zeros(max(capacity, 1) * 32, dtype=torch.uint8).pin_memory()
        else:
            buf = torch.zeros(max(capacity, 1) * 32, dtype=torch.uint8, device="cuda")
        cnt = loc.localize(fr, cam, threshold, buf, capacity)
        torch.cuda.synchronize()
        status = loc.check()
        found = int(cnt.value)
        em = P.emitters_to_numpy(buf, min(found, capacity))
        launches = loc.launch_count()
    if return_status:
        return em, found, status, launches
    assert status == P.OK
    assert found == len(em)
    return em


_ORACLE_CACHE = {}


def oracle_run(key, spec, weights, frames, cam_kw, dump_trunk=False):
    """Oracle forward (cached per test session by `key`)."""
    if key in _ORACLE_CACHE:
        return _ORACLE_CACHE[key]
    net = O.net_from_spec(spec)
    cam = O.make_camera(**cam_kw)
    res = O.forward_maps(net, weights, frames, cam, dump_trunk=dump_trunk)
    out = (net, cam) + (res if dump_trunk else (res, None))
    _ORACLE_CACHE[key] = out
    return out


def activated(spec, o):
    """The 'raw output maps' of the parity gate from pre-activation maps (float64 numpy math on
    whichever side's o): p, xy_scale*tanh, tanh (z), softplus (N, bg)."""
    o = np.asarray(o, dtype=np.float64)
    a = np.empty_like(o)
    nh = spec.head_channels
    a[:, 0] = 1.0 / (1.0 + np.exp(-o[:, 0]))
    a[:, 1] = spec.xy_scale * np.tanh(o[:, 1])
    a[:, 2] = spec.xy_scale * np.tanh(o[:, 2])
    h = 3
    if nh == 6:
        a[:, 3] = np.tanh(o[:, 3])
        h = 4
    for k in (h, h + 1):
        a[:, k] = np.maximum(o[:, k], 0) + np.log1p(np.exp(-np.abs(o[:, k])))
    return a


def contested_mask(p, threshold, tol):
    """Contested set of DESIGN.md: |p - thr| <= 0.02, or within 2*tol of a 3x3 neighbour
    (computed from the ORACLE's probability map p [n][H][W])."""
    n, H, W = p.shape
    c = np.abs(p - threshold) <= 0.02
    pad = np.full((n, H + 2, W + 2), np.inf)
    pad[:, 1:-1, 1:-1] = p
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            if dy == 0 and dx == 0:
                continue
            nb = pad[:, 1 + dy:H + 1 + dy, 1 + dx:W + 1 + dx]
            c |= np.abs(p - nb) <= 2 * tol
    return c


def parity_gate(spec, o_oracle, em_oracle, em_gpu, threshold, tol, pixel_size_nm, H, W,
                frame_offset=0):
    """Apply the gate; returns a dict of statistics (and asserts the hard conditions)."""
    p = 1.0 / (1.0 + np.exp(-np.asarray(o_oracle[:, 0], dtype=np.float64)))
    cm = contested_mask(p, threshold, tol)
    def key(em):
        return {(int(f) - frame_offset, int(q)) for f, q in zip(em["frame"], em["pix"])}
    so, sg = key(em_oracle), key(em_gpu)
    is_cont = lambda k: bool(cm[k[0]].ravel()[k[1]])
    so_u = {k for k in so if not is_cont(k)}
    sg_u = {k for k in sg if not is_cont(k)}
    assert so_u == sg_u, (f"uncontested detections differ: oracle-only {sorted(so_u - sg_u)[:5]}, "
                          f"gpu-only {sorted(sg_u - so_u)[:5]}")
    # matched pairs (contested or not): sub-pixel agreement
    go = {(int(e["frame"]) - frame_offset, int(e["pix"])): e for e in em_oracle}
    gg = {(int(e["frame"]) - frame_offset, int(e["pix"])): e for e in em_gpu}
    common = sorted(so & sg)
    dmax = {"x_px": 0.0, "y_px": 0.0, "p": 0.0, "rel_N": 0.0, "rel_bg": 0.0, "z_rel": 0.0}
    for k in common:
        a, b = go[k], gg[k]
        dmax["x_px"] = max(dmax["x_px"], abs(a["x_nm"] - b["x_nm"]) / pixel_size_nm)
        dmax["y_px"] = max(dmax["y_px"], abs(a["y_nm"] - b["y_nm"]) / pixel_size_nm)
        dmax["p"] = max(dmax["p"], abs(a["p"] - b["p"]))
        dmax["rel_N"] = max(dmax["rel_N"], abs(a["photons"] - b["photons"]) / max(abs(a["photons"]), 1e-9))
        dmax["rel_bg"] = max(dmax["rel_bg"], abs(a["bg"] - b["bg"]) / max(abs(a["bg"]), 1e-9))
        dmax["z_rel"] = max(dmax["z_rel"], abs(a["z_nm"] - b["z_nm"]) / max(spec.z_scale_nm, 1e-9))
    assert dmax["x_px"] <= 0.02 and dmax["y_px"] <= 0.02, dmax
    assert dmax["p"] <= tol, dmax
    n_cont = sum(1 for k in so if is_cont(k))
    return {"oracle": len(so), "gpu": len(sg), "matched": len(common),
            "contested_frac": n_cont / max(len(so), 1), "flipped": len(so ^ sg), **dmax}


def cam_kwargs(fs):
    return dict(pixel_size_nm=fs.pixel_size_nm, offset=fs.offset, gain=fs.gain,
                offset_map=fs.offset_map, gain_map=fs.gain_map)
