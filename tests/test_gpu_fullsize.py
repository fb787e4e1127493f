"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default
micro-batch, frames in a pinned host ring, emitter list written back to pinned host memory,
write-back batches where the config has them): sampled frames against the oracle, plus
properties that hold for every frame (the stack cycles a set of distinct frames, so frame f
and frame f + k must give the same detections; no two detections are 8-adjacent).
"""
import numpy as np
import pytest

from oracle import oracle as O
from smlm_synth import get_config, make_frames, make_weights
import paper_2410_02314_b200 as P
import gpu_util as G

pytestmark = pytest.mark.gpu


def _stack(cfg, n, k):
    fs = make_frames(cfg, k)
    reps = (n + k - 1) // k
    return fs, np.ascontiguousarray(np.concatenate([fs.frames] * reps)[:n])


def _check_cycle_and_adjacency(em, n, k, W):
    order = np.lexsort((em["pix"], em["frame"]))
    em = em[order]
    per = [em[em["frame"] == f] for f in range(min(k, n))]
    # every frame f >= k repeats frame f - k
    bounds = np.searchsorted(em["frame"], np.arange(n + 1))
    for f in range(k, n):
        a = em[bounds[f]:bounds[f + 1]]
        b = per[f % k]
        assert len(a) == len(b) and np.array_equal(a["pix"], b["pix"]), f
        for key in ("x_nm", "y_nm", "photons", "bg", "p"):
            assert np.array_equal(a[key], b[key]), (f, key)
    # no two detections of a frame are 8-adjacent (property of the rule, G8)
    for b in per[:4]:
        ys, xs = b["pix"] // W, b["pix"] % W
        grid = np.zeros((ys.max() + 3, W + 2), dtype=np.int32)
        grid[ys + 1, xs + 1] = 1
        nb = sum(np.roll(np.roll(grid, dy, 0), dx, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1))
        assert int((nb * grid).max()) == 1
    return em


def _oracle_gate(name, cfg, w, fs, em, sample, tol, H, W, max_contested=0.6):
    """Sampled frames of the production list against the oracle.  The contested set is built
    from the p-map error MEASURED on the same distinct frames (map export), see gpu_util."""
    ck = G.cam_kwargs(fs)
    net = O.net_from_spec(cfg.net)
    cam = O.make_camera(**ck)
    k = len(fs.frames)
    distinct = sorted({f % k for f in sample})
    o = {j: O.forward_maps(net, w, fs.frames[j:j + 1], cam) for j in distinct}
    og = G.gpu_forward_maps(cfg.net, w, np.ascontiguousarray(fs.frames[distinct]), ck)
    dp = {j: G.p_error(o[j], og[i:i + 1]) for i, j in enumerate(distinct)}
    stats = []
    for f in sample:
        em_o = O.postprocess(net, o[f % k], cam, cfg.threshold)
        em_o["frame"] += f
        em_g = em[em["frame"] == f]
        st = G.parity_gate(cfg.net, o[f % k], em_o, em_g, cfg.threshold, tol, fs.pixel_size_nm, H, W,
                           frame_offset=f, dp_measured=dp[f % k], o_gpu=og[distinct.index(f % k)][None])
        st["frame"] = f
        assert st["contested_frac_local"] <= max_contested and st["uncontested_local"] >= 100, st
        stats.append(st)
    G.record(name, gates=stats)
    return stats


def test_cfg1_full_1000_frames_pinned_ring_sampled_against_oracle():
    cfg = get_config(1)
    n, k = cfg.frames.n_frames, 16
    fs, frames = _stack(cfg, n, k)
    w = make_weights(cfg)
    cap = n * 4 * cfg.frames.emitters_per_frame
    em = G.gpu_localize(cfg.net, w, frames, G.cam_kwargs(fs), cfg.threshold, capacity=cap,
                        host_frames=True, host_out=True)
    em = _check_cycle_and_adjacency(em, n, k, 256)
    _oracle_gate("cfg1_full_1000_frames", cfg, w, fs, em, (0, 63, 64, 500, 999), 2e-2, 256, 256)


def test_cfg4_stream_10000_frames_writeback_256_sampled_against_oracle():
    """cfg 4 at its full size and launch configuration: 10 000 frames from a pinned host ring,
    emitter list written back every 256 frames (40 write-back batches)."""
    cfg = get_config(4)
    n, k = cfg.frames.n_frames, 8
    fs, frames = _stack(cfg, n, k)
    w = make_weights(cfg, "st")        # sharp p-map peaks (reading G28): the index gate covers >= 85 % of the detections
    cap = int(n * 1.5 * cfg.frames.emitters_per_frame)
    em = G.gpu_localize(cfg.net, w, frames, G.cam_kwargs(fs), cfg.threshold, capacity=cap,
                        host_frames=True, host_out=True, writeback_frames=cfg.writeback_batch)
    em = _check_cycle_and_adjacency(em, n, k, 256)
    _oracle_gate("cfg4_stream_10000_frames", cfg, w, fs, em, (0, 255, 256, 2559, 9999), 2e-2, 256, 256,
                 max_contested=0.15)


def test_cfg2_512x512_six_heads_sampled_against_oracle():
    cfg = get_config(2)
    n, k = 96, 2
    fs, frames = _stack(cfg, n, k)
    w = make_weights(cfg)
    cap = n * 3 * cfg.frames.emitters_per_frame
    em = G.gpu_localize(cfg.net, w, frames, G.cam_kwargs(fs), cfg.threshold, capacity=cap,
                        host_frames=True, host_out=True)
    em = _check_cycle_and_adjacency(em, n, k, 512)
    _oracle_gate("cfg2_full_frames", cfg, w, fs, em, (0, 95), 2e-2, 512, 512)


def test_cfg3_2048_tiled_sampled_rows_against_oracle_crop():
    """cfg 3: one full 2048x2048 frame through 512x512 tiles with per-pixel camera maps.  The
    oracle (which never tiles) runs on a 700x700 crop that covers a 2x2 tile crossing; inside
    the crop, at least radius+1 = 47 px from the crop's inner edges, both see the same
    receptive fields, so detections there must agree (reading G15)."""
    cfg = get_config(3)
    fs = make_frames(cfg, 1)
    w = make_weights(cfg)
    H = W = 2048
    ck = G.cam_kwargs(fs)
    frames = np.ascontiguousarray(np.concatenate([fs.frames, fs.frames]))
    lists = {}
    # NONE: the library default, 606 x 606 windows (layer pairs on 5-CTA clusters).  ROW: the shape
    # bench.py times for cfg 3, windows of 606 rows x the whole 2048-pixel width, one layer per kernel.
    for merge in (P.TILE_MERGE_NONE, P.TILE_MERGE_ROW):
        em = G.gpu_localize(cfg.net, w, frames, ck, cfg.threshold, capacity=2 * 4 * cfg.frames.emitters_per_frame,
                            host_frames=True, host_out=True, tile=cfg.tile, tile_merge=merge)
        a, b = em[em["frame"] == 0], em[em["frame"] == 1]
        assert len(a) > 1000 and np.array_equal(a["pix"], b["pix"]) and np.array_equal(a["x_nm"], b["x_nm"])
        lists[merge] = a
    # the two window shapes compute every owned pixel from the same receptive field
    assert lists[P.TILE_MERGE_NONE].tobytes() == lists[P.TILE_MERGE_ROW].tobytes()
    # crop with its origin at the frame origin: rows/cols 0..699 (the frame border keeps its
    # zero padding, the inner edges lose 47 px)
    S, M = 700, 47
    crop = np.ascontiguousarray(fs.frames[:, :S, :S])
    ckc = dict(ck, offset_map=np.ascontiguousarray(fs.offset_map[:S, :S]),
               gain_map=np.ascontiguousarray(fs.gain_map[:S, :S]))
    net = O.net_from_spec(cfg.net)
    cam = O.make_camera(**ckc)
    o = O.forward_maps(net, w, crop, cam)
    em_o = O.postprocess(net, o, cam, cfg.threshold)
    inner = lambda y, x: (y < S - M) & (x < S - M)
    yo, xo = em_o["pix"] // S, em_o["pix"] % S
    em_o = em_o[inner(yo, xo)]
    a = lists[P.TILE_MERGE_ROW]                    # the timed shape against the oracle (NONE is byte-identical)
    ya, xa = a["pix"] // W, a["pix"] % W
    ag = a[inner(ya, xa)].copy()
    ag["pix"] = (ya[inner(ya, xa)] * S + xa[inner(ya, xa)]).astype(np.int32)
    # p-map error measured on the same crop through the map export (valid where the
    # receptive field lies inside the crop: the same inner region)
    og = G.gpu_forward_maps(cfg.net, w, crop, ckc)
    dp = G.p_error(o[:, :, :S - M + 1, :S - M + 1], og[:, :, :S - M + 1, :S - M + 1])
    # (the local bound needs maps that are comparable everywhere: outside the inner region the
    # crop's own border changes the oracle's maps, and no detection is compared there)
    og_in = o.astype(np.float32).copy()
    og_in[:, :, :S - M + 1, :S - M + 1] = og[:, :, :S - M + 1, :S - M + 1]
    st = G.parity_gate(cfg.net, o, em_o, ag, cfg.threshold, 2e-2, fs.pixel_size_nm, S, S, dp_measured=dp,
                       o_gpu=og_in)
    G.record("cfg3_2048_tiled_vs_oracle_crop", gate=st, shapes="tile_merge ROW (timed) == NONE byte for byte")
    assert st["oracle"] > 1000 and st["contested_frac_local"] <= 0.6 and st["uncontested_local"] >= 100, st
