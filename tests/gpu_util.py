"""Helpers shared by the GPU parity tests: run the CUDA library through its C ABI binding,
run the oracle on the same seeded inputs, and apply the parity gate of DESIGN.md."""
from __future__ import annotations

import json
import os

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


def contested_mask(p, threshold, dp, band=None):
    """Contested set of DESIGN.md section 5, computed from the ORACLE's probability map
    p [n][H][W]: |p - thr| <= band, or within 2*dp of a 3x3 neighbour.  dp is a bound that the
    GPU's p-map satisfies (|p_gpu - p_oracle| <= dp everywhere): the decision at a pixel is a
    pure function of its 3x3 logits, so outside this set the two sides cannot decide
    differently."""
    n, H, W = p.shape
    c = np.abs(p - threshold) <= (dp if band is None else band)
    pad = np.full((n, H + 2, W + 2), np.inf)
    pad[:, 1:-1, 1:-1] = p
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            if dy == 0 and dx == 0:
                continue
            nb = pad[:, 1 + dy:H + 1 + dy, 1 + dx:W + 1 + dx]
            c |= np.abs(p - nb) <= 2 * dp
    return c


def p_error(o_oracle, o_gpu):
    """max |p_gpu - p_oracle| over all pixels (float64 sigmoid of both pre-activation maps)."""
    a = 1.0 / (1.0 + np.exp(-np.asarray(o_oracle[:, 0], dtype=np.float64)))
    b = 1.0 / (1.0 + np.exp(-np.asarray(o_gpu[:, 0], dtype=np.float64)))
    return float(np.max(np.abs(a - b)))


def local_contested_mask(p, p_gpu, threshold):
    """The same theorem with a LOCAL bound: e = |p_gpu - p_oracle| per pixel, E(q) = max of e
    over the 3x3 neighbourhood of q.  Both q and each neighbour m are off by at most E(q), so
    the decision at q cannot differ unless |p_q - p_m| <= 2 E(q) for some m or
    |p_q - thr| <= E(q).  Tighter than the global bound: one outlier pixel no longer widens
    the contested set of the whole frame."""
    n, H, W = p.shape
    e = np.abs(p_gpu - p)
    epad = np.zeros((n, H + 2, W + 2))
    epad[:, 1:-1, 1:-1] = e
    E = np.zeros_like(e)
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            E = np.maximum(E, epad[:, 1 + dy:H + 1 + dy, 1 + dx:W + 1 + dx])
    E = E * (1 + 1e-9) + 1e-12
    c = np.abs(p - threshold) <= E
    pad = np.full((n, H + 2, W + 2), np.inf)
    pad[:, 1:-1, 1:-1] = p
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            if dy == 0 and dx == 0:
                continue
            c |= np.abs(p - pad[:, 1 + dy:H + 1 + dy, 1 + dx:W + 1 + dx]) <= 2 * E
    return c


def parity_gate(spec, o_oracle, em_oracle, em_gpu, threshold, tol, pixel_size_nm, H, W,
                frame_offset=0, dp_measured=None, check_tol=True, o_gpu=None):
    """Apply the gate; returns a dict of statistics (and asserts the hard conditions).

    dp_measured: max |p_gpu - p_oracle| measured on the maps of this very run.  When given, it
    must be <= tol (unless check_tol is False: the high-contrast weights in bf16), and the
    contested set is built from it - 2 x the measured error around neighbours, the measured
    error (at most BASELINE.json's 0.02) around the threshold - instead of from the
    tolerance, so that the index gate covers every detection the theorem allows it to cover.
    Without it the set is built from tol and 0.02 (the fp32 cases, whose tol is tiny).
    o_gpu: the GPU's pre-activation maps of the same frames (map export).  When given, the
    gate is applied a second time with the local bound of local_contested_mask."""
    p = 1.0 / (1.0 + np.exp(-np.asarray(o_oracle[:, 0], dtype=np.float64)))
    if dp_measured is None:
        cm = contested_mask(p, threshold, tol, band=0.02)
    else:
        if check_tol:
            assert dp_measured <= tol, f"p-map error {dp_measured} above the tolerance {tol}"
        dp = dp_measured * (1 + 1e-9) + 1e-12
        cm = contested_mask(p, threshold, dp, band=min(dp, 0.02) if check_tol else dp)
    def key(em):
        return {(int(f) - frame_offset, int(q)) for f, q in zip(em["frame"], em["pix"])}
    so, sg = key(em_oracle), key(em_gpu)

    def apply(mask, what):
        is_c = lambda k: bool(mask[k[0]].ravel()[k[1]])
        so_u = {k for k in so if not is_c(k)}
        sg_u = {k for k in sg if not is_c(k)}
        assert so_u == sg_u, (f"{what}: uncontested detections differ: oracle-only "
                              f"{sorted(so_u - sg_u)[:5]}, gpu-only {sorted(sg_u - so_u)[:5]}")
        return len(so_u), 1.0 - len(so_u) / max(len(so), 1)

    n_unc, frac = apply(cm, "global bound")
    local = {}
    if o_gpu is not None:
        pg = 1.0 / (1.0 + np.exp(-np.asarray(o_gpu[:, 0], dtype=np.float64)))
        n_unc_l, frac_l = apply(local_contested_mask(p, pg, threshold), "local bound")
        local = {"uncontested_local": n_unc_l, "contested_frac_local": frac_l}
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
    if check_tol:
        assert dmax["x_px"] <= 0.02 and dmax["y_px"] <= 0.02, dmax
        assert dmax["p"] <= tol, dmax
    return {"oracle": len(so), "gpu": len(sg), "matched": len(common), "uncontested": n_unc,
            "contested_frac": frac, "flipped": len(so ^ sg), "dp_measured": dp_measured, **local,
            **{k: float(v) for k, v in dmax.items()}}


# ---------------------------------------------------------------------------- parity record
# Every gate run appends its statistics to one JSON file ("a vacuous gate must be visible").  The
# file goes where SMLM_PARITY_RECORD points (a GPU run sets it to a path that travels back, and a
# summary of it is committed under profiles/), else to the system's temporary directory.
import tempfile

_RECORD_PATH = os.environ.get("SMLM_PARITY_RECORD") or os.path.join(tempfile.gettempdir(), "smlm_parity_record.json")
_RECORDS = {}


def record(test, **stats):
    def plain(v):
        if isinstance(v, dict):
            return {k: plain(x) for k, x in v.items()}
        if isinstance(v, (list, tuple)):
            return [plain(x) for x in v]
        if isinstance(v, (np.floating, np.integer)):
            return v.item()
        if isinstance(v, np.ndarray):
            return v.tolist()
        return v
    _RECORDS[test] = plain(stats)
    try:
        os.makedirs(os.path.dirname(os.path.abspath(_RECORD_PATH)), exist_ok=True)
        with open(_RECORD_PATH, "w", encoding="utf-8") as fh:
            json.dump({"written_by": "tests/gpu_util.py record() during `pytest tests -m gpu`",
                       "records": _RECORDS}, fh, indent=1, sort_keys=True)
    except OSError:
        pass


def head_errors(spec, o_oracle, o_gpu):
    """Per-head max |activated(gpu) - activated(oracle)| (the 'raw output maps' of the gate)."""
    nh = spec.head_channels
    d = np.abs(activated(spec, o_gpu) - activated(spec, o_oracle))
    return d.transpose(1, 0, 2, 3).reshape(nh, -1).max(axis=1)


def cam_kwargs(fs):
    return dict(pixel_size_nm=fs.pixel_size_nm, offset=fs.offset, gain=fs.gain,
                offset_map=fs.offset_map, gain_map=fs.gain_map)
