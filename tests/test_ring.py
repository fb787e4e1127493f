"""The disk -> pinned-ring loader (include/smlm.h smlm_ring_*).

CPU part: the reader threads and the slot hand-over, on a pageable ring (no device needed).
GPU part: smlm_localize_ring over a frame file must give the emitter list of the all-in-memory
smlm_localize call, bit by bit."""
import os

import numpy as np
import pytest

import paper_2410_02314_b200 as P


def _write(tmp_path, frames, offset=0):
    path = os.path.join(tmp_path, "frames.u16")
    with open(path, "wb") as fh:
        fh.write(b"\0" * offset)
        fh.write(np.ascontiguousarray(frames, dtype="<u2").tobytes())
    return path


@pytest.mark.parametrize("n,chunk,slots,threads,offset", [(23, 5, 2, 3, 0), (8, 8, 2, 1, 64), (40, 3, 4, 4, 10),
                                                          (1, 7, 3, 2, 0), (0, 4, 2, 1, 0)])
def test_ring_delivers_the_file_in_order(tmp_path, n, chunk, slots, threads, offset):
    rng = np.random.default_rng(n * 100 + chunk)
    H, W = 9, 13
    frames = rng.integers(0, 65536, size=(n, H, W)).astype(np.uint16)
    path = _write(str(tmp_path), frames, offset)
    with P.Ring(path, n, H, W, chunk, n_slots=slots, n_threads=threads, byte_offset=offset, pageable=True) as ring:
        seen = 0
        held = []
        while True:
            arr, first = ring.acquire()
            if arr is None:
                break
            assert first == seen and arr.shape[0] == min(chunk, n - seen)
            assert np.array_equal(arr, frames[first:first + arr.shape[0]])
            seen += arr.shape[0]
            held.append(first)
            if len(held) == slots:              # hold every slot once: the readers must wait, not overrun
                for f in held:
                    ring.release(f)
                held = []
        for f in held:
            ring.release(f)
        assert seen == n


def test_ring_refuses_bad_arguments(tmp_path):
    frames = np.zeros((4, 8, 8), np.uint16)
    path = _write(str(tmp_path), frames)
    with pytest.raises(P.SmlmError):
        P.Ring(path, 5, 8, 8, 2, pageable=True)                      # file shorter than 5 frames
    with pytest.raises(P.SmlmError):
        P.Ring(path + ".missing", 4, 8, 8, 2, pageable=True)
    with pytest.raises(P.SmlmError):
        P.Ring(path, 4, 8, 8, 2, n_slots=1, pageable=True)


@pytest.mark.gpu
@pytest.mark.parametrize("chunk,slots,threads,kw", [(7, 3, 2, {}), (16, 2, 4, dict(writeback_frames=9)),
                                                    (5, 4, 1, dict(micro_batch=3))])
def test_localize_ring_equals_in_memory_localize(tmp_path, chunk, slots, threads, kw):
    import torch
    import gpu_util as G
    from smlm_synth import get_config, make_frames, make_weights
    cfg = get_config(0)
    fs = make_frames(cfg, 8)
    frames = np.ascontiguousarray(np.concatenate([fs.frames] * 7)[:53])
    w = make_weights(cfg)
    ck = G.cam_kwargs(fs)
    ref = G.gpu_localize(cfg.net, w, frames, ck, cfg.threshold, host_frames=True, host_out=True, **kw)
    path = _write(str(tmp_path), frames)
    n, H, W = frames.shape
    cap = n * ((H + 1) // 2) * ((W + 1) // 2)
    with P.Localizer(P.desc_from_spec(cfg.net, **kw), w) as loc, \
            P.Ring(path, n, H, W, chunk, n_slots=slots, n_threads=threads) as ring:
        buf = torch.zeros(cap * 32, dtype=torch.uint8).pin_memory()
        for _ in range(2):                                           # a ring serves several passes
            cnt = loc.localize_ring(ring, loc.camera(**ck), cfg.threshold, buf, cap)
            torch.cuda.synchronize()
            assert loc.check() == P.OK, loc.last_error()
            em = P.emitters_to_numpy(buf, cnt.value)
            assert len(em) == len(ref) and em.tobytes() == ref.tobytes()
        with P.Ring(path, n, H, W, chunk, pageable=True) as bad, pytest.raises(P.SmlmError):
            loc.localize_ring(bad, loc.camera(**ck), cfg.threshold, buf, cap)


@pytest.mark.gpu
@pytest.mark.timeout(180)
def test_localize_ring_back_to_back_calls_without_sync(tmp_path):
    """The host enqueues several smlm_localize_ring calls before the GPU has finished the first:
    each call rewinds the ring while the previous pass's H2D copies and slot releases are still
    pending.  The rewind must wait for them (a late release of old chunk k used to free the slot
    holding new chunk k, and the host then waited for that chunk forever; seen as a hung
    bench.py --disk).  Every call must give the in-memory result."""
    import torch
    import gpu_util as G
    from smlm_synth import get_config, make_frames, make_weights
    cfg = get_config(1)
    fs = make_frames(cfg, 4)
    frames = np.ascontiguousarray(np.concatenate([fs.frames] * 16))           # 64 frames of 256 x 256
    w = make_weights(cfg)
    ck = G.cam_kwargs(fs)
    ref = G.gpu_localize(cfg.net, w, frames, ck, cfg.threshold, host_frames=True, host_out=True)
    path = _write(str(tmp_path), frames)
    n, H, W = frames.shape
    cap = n * 2048
    calls = 12
    with P.Localizer(P.desc_from_spec(cfg.net), w) as loc, P.Ring(path, n, H, W, 16, n_slots=2, n_threads=3) as ring:
        stream = torch.cuda.Stream()
        bufs = [torch.zeros(cap * 32, dtype=torch.uint8).pin_memory() for _ in range(calls)]
        cam = loc.camera(**ck)
        cnts = [loc.localize_ring(ring, cam, cfg.threshold, b, cap, stream=stream) for b in bufs]
        torch.cuda.synchronize()
        assert loc.check() == P.OK, loc.last_error()
        for b, c in zip(bufs, cnts):
            em = P.emitters_to_numpy(b, c.value)
            assert len(em) == len(ref) and em.tobytes() == ref.tobytes()


def test_rewind_of_a_partly_consumed_ring_delivers_every_chunk_once(tmp_path):
    """A pass abandoned part-way (chunks taken and released by hand, then a rewind): the readers
    hold assignments for later chunks and wait for slots.  None of those claims may survive the
    rewind - a survivor would read its chunk a second time into a slot of the new pass (wrong
    frames, or a consumer that waits forever).  8 chunks, 2 slots, 3 readers, many repeats."""
    rng = np.random.default_rng(5)
    n, chunk, H, W = 8 * 3, 3, 5, 7
    frames = rng.integers(0, 65536, size=(n, H, W)).astype(np.uint16)
    path = _write(str(tmp_path), frames)
    with P.Ring(path, n, H, W, chunk, n_slots=2, n_threads=3, pageable=True) as ring:
        for it in range(400):
            for _ in range((2, 0, 5, 1, 8, 3)[it % 6]):          # abandon the pass after this many chunks
                arr, first = ring.acquire()
                if arr is None:
                    break
                ring.release(first)
            ring.rewind()
            seen = 0
            while True:
                arr, first = ring.acquire()
                if arr is None:
                    break
                assert first == seen, (it, first, seen)
                assert np.array_equal(arr, frames[first:first + arr.shape[0]]), (it, first)
                seen += arr.shape[0]
                ring.release(first)
            assert seen == n
            ring.rewind()
