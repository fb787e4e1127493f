#!/usr/bin/env python
"""Benchmark of the hot path (BASELINE.json metric: frames/s and emitters/s at 256x256 on one
B200, device-timed; % of tensor / HBM peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1]

One "step" = one smlm_localize call over the whole synthetic stack of the config (every row
of the hot path: preload ring -> K1 stem -> K2 x L dilated convs -> K3 heads + post).
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from smlm_synth import get_config, make_frames, make_weights  # noqa: E402

METRIC = "frames_per_s_256x256"
UNIT = "frames/s"
REPEATS = 3                 # timed windows per path; the median one is reported
DISTINCT_FRAMES = 128       # generated once, cycled to the config's frame count (throughput is data-independent)
# /opt/skills/guides/B200_PROFILING.md, "Peaks and the roofline denominators": "FALLBACK, only if that file
# is absent ...: 6.65 TB/s and 1.59 PFLOP/s ... (1.59 is the burst figure; sustained it settles near 1.4 PFLOP/s)".
# A line computed from these says peak_source "fallback".
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p, "r", encoding="utf-8") as fh:
            d = json.load(fh)
        return d, "measured"
    return dict(FALLBACK_PEAKS), "fallback"


def lookup_traffic(cfg, C, views, bound, pair=False, fusion="auto"):
    """(bytes per full-size launch, provenance) of the dominant K2 kernel from profiles/traffic_r2.json."""
    path = os.path.join(ROOT, "profiles", "traffic_r2.json")
    if bound != "tensor" or not os.path.exists(path):
        return None, "no capture"
    with open(path, "r", encoding="utf-8") as fh:
        doc = json.load(fh)
    wl = {4: "cfg1"}.get(cfg.index, f"cfg{cfg.index}")        # cfg 4 launches are cfg 1's (same net, same shape)
    cap = doc.get("captures", {}).get(f"{wl}/views{views}")
    if not cap:
        return None, f"no capture for {wl}/views{views} in profiles/traffic_r2.json"
    name = f"conv_umma_kernel<{C},-,->"
    if pair:   # cta_group::2 where a row has an even number of segments (conv_pair.cu)
        name = f"conv_pair_kernel<{C},-,-,{'cg2' if (-(-cfg.frames.width // 128)) % 2 == 0 and fusion != 'pairs1' else 'cg1'}>"
    k = cap["per_kernel_mean"].get(name)
    if not k:
        return None, f"capture {wl}/views{views} holds no {name} launch"
    note = (f"profiles/traffic_r2.json {wl}/views{views}: mean of {k['n']} {name} launches of {views} views "
            f"(ncu --set full, {cap.get('source', '')}); the HEAD launch and the tail launch of a step are listed "
            f"there separately")
    return k["dram_bytes"], note


def workload(cfg, n_frames=None):
    n = cfg.frames.n_frames if n_frames is None else n_frames
    # bounded generation time: at most 2^25 distinct pixels (cfg 3: 8 distinct 2048x2048 frames)
    k = min(DISTINCT_FRAMES, n, max(4, (1 << 25) // (cfg.frames.height * cfg.frames.width)))
    fs = make_frames(cfg, k)
    reps = (n + k - 1) // k
    frames = np.concatenate([fs.frames] * reps)[:n]
    return fs, np.ascontiguousarray(frames)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index
        self.rows = []
        self.stop_flag = threading.Event()
        # NVML in-process (nvidia_ml_py) where it loads: a query costs microseconds and spawns
        # nothing.  Forking nvidia-smi ten times a second inside the timed region perturbed the
        # measurement itself (the first run on a fresh box, with the binary cold, by ~5 %).
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            phys = index
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            if vis and all(v.strip().isdigit() for v in vis.split(",")) and index < len(vis.split(",")):
                phys = int(vis.split(",")[index])
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def sample_nvml(self):
        n, h = self.nvml, self.handle
        sm = float(n.nvmlDeviceGetClockInfo(h, n.NVML_CLOCK_SM))
        pw = n.nvmlDeviceGetPowerUsage(h) / 1000.0
        try:
            rs = int(n.nvmlDeviceGetCurrentClocksEventReasons(h))
        except Exception:
            rs = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(h))
        flag = lambda bit: "Active" if rs & bit else "Not Active"
        return [str(sm), str(self.max_sm), "%.2f" % pw,
                flag(getattr(n, "nvmlClocksThrottleReasonHwSlowdown", 0x8)),
                flag(getattr(n, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40)),
                flag(getattr(n, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20)),
                flag(getattr(n, "nvmlClocksThrottleReasonSwPowerCap", 0x4))]

    def run(self):
        while not self.stop_flag.is_set():
            try:
                if self.nvml is not None:
                    self.rows.append(self.sample_nvml())
                else:
                    out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                    parts = [p.strip() for p in out.strip().split(",")]
                    if len(parts) >= 7:
                        self.rows.append(parts)
            except Exception:
                pass
            self.stop_flag.wait(0.05 if self.nvml is not None else 0.1)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows)
        reasons = []
        for i, name in enumerate(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")):
            if any(r[3 + i].lower().startswith("active") for r in self.rows):
                reasons.append(name)
        pw = max(float(r[2]) for r in self.rows if r[2].replace(".", "", 1).isdigit())
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "power_w_max": pw,
                "samples": len(self.rows), "reasons": reasons,
                "source": "NVML (nvidia_ml_py), every 50 ms" if self.nvml is not None else "nvidia-smi, every 100 ms"}


def oracle_sample(cfg, fs, weights, n_sample):
    """The oracle as it stands, timed on this host's cores on the first n_sample frames."""
    from oracle import oracle as O
    net = O.net_from_spec(cfg.net)
    cam = O.make_camera(fs.pixel_size_nm, fs.offset, fs.gain, fs.offset_map, fs.gain_map)
    O.lib()
    t0 = time.perf_counter()
    em = O.localize(net, weights, fs.frames[:n_sample], cam, cfg.threshold)
    dt = time.perf_counter() - t0
    return n_sample / dt, len(em) / dt, O.threads(), dt


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    fs, _ = workload(cfg, n_frames=16)
    w = make_weights(cfg)
    # one step = a bounded sample: about 5e11 FLOP of oracle work (a few seconds on 16 cores)
    H, W = cfg.frames.height, cfg.frames.width
    n_sample = max(1, min(len(fs.frames), int(5e11 / (cfg.net.flop_per_px() * H * W))))
    for _ in range(args.warmup):
        oracle_sample(cfg, fs, w, 1)
    t_tot, frames = 0.0, 0
    cores = 1
    for _ in range(args.steps):
        fps, eps, cores, dt = oracle_sample(cfg, fs, w, n_sample)
        t_tot += dt
        frames += n_sample
    value = frames / t_tot
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": cfg.name, "H": cfg.frames.height, "W": cfg.frames.width,
                       "channels": cfg.net.channels, "layers": cfg.net.n_layers,
                       "frames_per_step": n_sample, "note": "fp64 CPU oracle on host cores, bounded sample"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{n_sample} frame(s) of {cfg.name} per step"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def dloc_flop_per_px(spec):
    """2 x MAC per full-resolution pixel (dloc.h): the DCD blocks and dec0 at full resolution,
    enc1 / dec1 at 1/4 of the pixels, enc2 at 1/16."""
    C = spec.c0
    f = 0.0
    for name, co, ci, k in spec.layers():
        scale = {"enc1": 0.25, "dec1": 0.25, "enc2": 1.0 / 16}.get(name, 1.0)
        f += 2.0 * co * ci * k * k * scale
    return f


def dloc_bytes_per_px(spec, elt=2):
    """Algorithmic HBM bytes of the timed convolution launches per full-resolution pixel: every
    launch reads its input channels and writes its output channels once (a
    dense-block layer re-reads the whole concatenation so far), 16-bit storage; enc1 / dec1 at 1/4 of
    the pixels, enc2 at 1/16; the heads write fp32 planes.  Stem, pool and upsample kernels are not
    among the timed launches."""
    b = 0.0
    for name, co, ci, k in spec.layers():
        if name == "stem":
            continue
        scale = {"enc1": 0.25, "dec1": 0.25, "enc2": 1.0 / 16}.get(name, 1.0)
        b += (ci * elt + co * (4 if name == "head" else elt)) * scale
    return b


def run_dloc(args, cfg):
    """The paper's own topology through dloc_localize: same step, timing and JSON contract as
    the headline path (one step = one call over the whole stack; value device-resident, e2e
    from pinned host frames to a pinned host list)."""
    import dataclasses
    import torch
    import paper_2410_02314_b200 as P
    from paper_2410_02314_b200 import dloc_binding as DB
    from smlm_synth import DlocSpec, dloc_he_normal_blob
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    torch.cuda.set_device(0)
    spec = DlocSpec(precision=args.precision or "bf16")
    n_frames = args.frames or cfg.frames.n_frames
    fs, frames = workload(cfg, n_frames)
    H, W = frames.shape[1:]
    weights = dloc_he_normal_blob(spec, 7, head_gain=0.5)
    conv_impl = {"auto": P.CONV_AUTO, "tcgen05": P.CONV_TCGEN05, "direct": P.CONV_DIRECT}[args.conv_impl]
    loc = DB.DlocLocalizer(DB.dloc_desc_from_spec(spec, micro_batch=args.micro_batch, conv_impl=conv_impl), weights)
    cap = n_frames * ((H + 1) // 2) * ((W + 1) // 2)
    cap = min(cap, int(n_frames * max(8 * cfg.frames.emitters_per_frame, 4096)))
    cam = loc.camera(fs.pixel_size_nm, fs.offset, fs.gain)
    frames_host = torch.from_numpy(frames).pin_memory()
    frames_dev = frames_host.cuda()
    out_dev = torch.zeros(cap * 48, dtype=torch.uint8, device="cuda")
    out_host = torch.zeros(cap * 48, dtype=torch.uint8).pin_memory()
    stream = torch.cuda.Stream()
    thr = 0.5

    def timed(frames_t, out_t, steps, kernel_timing=False):
        loc.kernel_timing(kernel_timing)
        torch.cuda.synchronize()
        l0 = loc.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        counts = []
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(steps):
                counts.append(loc.localize(frames_t, cam, thr, out_t, cap, stream=stream))
            e1.record(stream)
        torch.cuda.synchronize()
        if loc.check() != P.OK:
            raise SystemExit(f"dloc_check: {loc.check()} {loc.last_error()}")
        kt = loc.conv_time_ms() if kernel_timing else None
        loc.kernel_timing(False)
        return e0.elapsed_time(e1), [int(getattr(c, "value", c)) for c in counts], loc.launch_count() - l0, kt

    timed(frames_dev, out_dev, args.warmup)
    timed(frames_host, out_host, args.warmup)
    sampler = ClockSampler(0)
    sampler.start()
    ms, counts, launches, _ = timed(frames_dev, out_dev, args.steps)
    ms_e2e, counts_e2e, _, _ = timed(frames_host, out_host, args.steps)
    ms_rf, _, _, (conv_ms, conv_n) = timed(frames_dev, out_dev, args.steps, kernel_timing=True)
    sampler.stop_flag.set()
    sampler.join(timeout=2)
    peaks, peak_kind = load_peaks()
    fpp = dloc_flop_per_px(spec)
    stem_head = 2.0 * spec.c0 * spec.in_frames * 9 + 2.0 * spec.c0 * spec.head_channels   # not tensor-core work
    conv_flop = (fpp - stem_head) * H * W * n_frames * args.steps
    peak = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
    achieved = conv_flop / (conv_ms * 1e-3) / 1e12 if conv_ms > 0 else None
    roofline = None
    if achieved is not None:
        # which kernels ran the timed launches (dloc.cu: conv_impl AUTO = the row-chain kernel for every
        # convolution but dec1, whose 288 input channels go through the generic implicit GEMM)
        kernels = {"auto": "conv_chain_kernel (dense-block layers, 1x1 transitions, enc1, enc2, dec0, heads) + "
                           "conv_gen_umma_kernel (dec1)",
                   "tcgen05": "conv_gen_umma_kernel (every convolution but the stem)",
                   "direct": "conv_gen_direct_kernel (every convolution but the stem; CUDA cores)"}[args.conv_impl]
        tensor = {"achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                  "frac_of_burst": achieved / float(peaks["bf16_tflops"]),
                  "peak_source": f"{peak_kind} bf16_tflops_sustained (kernels timed inside a long step)"}
        gbs = dloc_bytes_per_px(spec, 4 if spec.precision == "fp32" else 2) * H * W * n_frames * args.steps \
            / (conv_ms * 1e-3) / 1e9
        hbm = {"achieved": gbs, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s", "frac": gbs / float(peaks["hbm_gbs"]),
               "peak_source": f"{peak_kind} hbm_gbs (copy bandwidth)",
               "bytes_per_px": dloc_bytes_per_px(spec, 4 if spec.precision == "fp32" else 2)}
        # the binding roof is the one the launches sit closer to: the dense-block launches move
        # 1 024 B/px per block and run at 88-100 % of the copy bandwidth
        if args.conv_impl == "direct" or spec.precision == "fp32":
            lead, bound = hbm if hbm["frac"] > 0.5 else tensor, "hbm" if hbm["frac"] > 0.5 else "alu"
        else:
            lead, bound = (hbm, "hbm") if hbm["frac"] >= tensor["frac"] else (tensor, "tensor")
        roofline = {"bound": bound, "kernel": kernels, **{k: lead[k] for k in ("achieved", "peak", "unit", "frac", "peak_source")},
                    "traffic": None, "traffic_source": "no ncu --set full capture of the whole launch set "
                                                       "(profiles/ holds one of the dense-block chain kernel)",
                    "against_tensor_peak": tensor, "against_hbm_peak": hbm,
                    "launches": conv_n, "avg_launch_ms": conv_ms / max(conv_n, 1), "share_of_step": conv_ms / ms_rf}
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import dloc as D
        from oracle import oracle as O
        ns = max(1, min(len(fs.frames), int(2.5e11 / (fpp * H * W))))    # ~15 s: this oracle runs at ~15 GFLOP/s
        ocam = O.make_camera(fs.pixel_size_nm, fs.offset, fs.gain)
        t0 = time.perf_counter()
        o = D.forward_maps(D.net_from_spec(spec), weights, fs.frames[:ns], ocam)
        em = D.postprocess(spec, o, ocam, thr)
        dt = time.perf_counter() - t0
        cpu = {"value": ns / dt, "unit": UNIT, "cores": O.threads(), "kind": "oracle",
               "sample": f"first {ns} frame(s), {dt:.1f} s (oracle/dloc_oracle.c)", "emitters_per_s": len(em) / dt}
    line = {"metric": METRIC, "value": n_frames * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": {"bf16": "bf16", "fp16": "f16"}.get(spec.precision, "f32"),
            "data": "synthetic",
            "config": {"workload": f"dloc_c{spec.c0}g{spec.growth}_b{spec.n_blocks}_on_{cfg.name}", "frames_per_step": n_frames,
                       "H": H, "W": W, "c0": spec.c0, "growth": spec.growth, "n_blocks": spec.n_blocks,
                       "dilations": list(spec.dilations), "head_channels": spec.head_channels,
                       "precision": spec.precision, "conv_impl": args.conv_impl, "flop_per_px": fpp,
                       "l2": "inputs larger than L2 (u16 stack + feature maps per step > 126 MB)",
                       "parallelism": "replicas x1"},
            "emitters_per_s": sum(counts) / (ms * 1e-3), "emitters_per_frame": sum(counts) / (n_frames * args.steps),
            "e2e": {"value": n_frames * args.steps / (ms_e2e * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(frames.nbytes), "d2h_bytes_per_step": int(counts_e2e[-1] * 48 + 8),
                    "ms_per_step": ms_e2e / args.steps, "exposed_copy_ms_per_step": (ms_e2e - ms) / args.steps},
            "gpu_launches": launches, "clocks": sampler.summary(), "roofline": roofline, "cpu_baseline": cpu,
            "tensor_frac_whole_step": (fpp * H * W * n_frames * args.steps / (ms * 1e-3) / 1e12)
                                      / float(peaks["bf16_tflops"])}
    print(json.dumps(line), flush=True)
    loc.close()
    return 0


OTHER_CONFIGS = {   # short device-resident runs appended to the default line (the driver's record then holds them too)
    "cfg2_3d_astig_512_bf16": ["--config", "2", "--frames", "96"],
    "cfg3_fov2048_tiled_bf16": ["--config", "3", "--frames", "8"],
    "cfg4_dense_stream_bf16": ["--config", "4", "--frames", "2560"],
    "dloc_on_cfg1": ["--net", "dloc", "--frames", "256"],
}


def other_configs(args):
    """Each of OTHER_CONFIGS as a child `bench.py` process after the headline's timed region (own
    process: own clocks sample, no shared device memory); its JSON line reduced to the judged keys."""
    import subprocess
    out = {}
    for name, extra in OTHER_CONFIGS.items():
        cmd = [sys.executable, os.path.abspath(__file__), *extra, "--steps", "3", "--warmup", "3", "--no-cpu-baseline",
               "--no-other-configs", "--weights", args.weights]
        try:
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
            d = json.loads(r.stdout.strip().splitlines()[-1])
            out[name] = {k: d.get(k) for k in ("value", "unit", "ms_per_step", "steps", "dtype", "config", "e2e", "gpu_launches",
                                               "clocks", "roofline", "io_kernels", "tensor_frac_whole_step", "emitters_per_frame")}
            out[name]["command"] = "python bench.py " + " ".join(cmd[2:])
        except Exception as ex:  # the headline line must still be printed
            out[name] = {"error": f"{type(ex).__name__}: {ex}"[:300]}
    return out


def _rank_entry(rank, world, port, argv):
    """One rank of a self-spawned run: the same environment torchrun would set."""
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), LOCAL_WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    rc = main(argv)
    if rc:
        raise SystemExit(rc)


def spawn_ranks(args, argv):
    """python bench.py --gpus N without torchrun: start N ranks, one per GPU (multi-GPU =
    independent replicas: the only communication is the barrier and the reduction of
    two scalars)."""
    import socket
    import torch
    import torch.multiprocessing as mp
    if not args.selftest_spawn and torch.cuda.device_count() < args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus}: only {torch.cuda.device_count()} CUDA device(s) visible")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    mp.spawn(_rank_entry, args=(args.gpus, port, argv), nprocs=args.gpus, join=True)
    return 0


def selftest_spawn(args, cfg):
    """Host logic of the N > 1 path on CPU (gloo): sharding + whole-job throughput."""
    import torch.distributed as dist
    from paper_2410_02314_b200.replicas import job_throughput, shard_frames
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    n = args.frames or cfg.frames.n_frames
    lo, hi = shard_frames(n, rank, world) if args.scaling == "strong" else (0, n)
    ms = 10.0 + rank                                   # synthetic device time: the slowest rank decides
    value, ms_max = job_throughput(hi - lo, ms, dist if world > 1 else None, "cpu")
    if rank == 0:
        print(json.dumps({"selftest": True, "n_gpus": world, "scaling": args.scaling, "value": value,
                          "ms_max": ms_max, "frames_rank0": hi - lo}), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0,
                    help="timed steps; default: 40 for cfg 0 / 1 (1.3 s, averages over the dips of the power governor), "
                         "5 / 3 / 4 for cfg 2 / 3 / 4, 5 for --net dloc")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--net", default="stack", choices=["stack", "dloc"],
                    help="stack: BASELINE.json's residual dilated stack (smlm.h, the headline); dloc: the paper's own "
                         "topology (dloc.h, SURVEY.md 8(f)-2: DCD dense blocks, dilations 2-4-8-16, two-stage U-Net, "
                         "ten heads) on the config's frames")
    ap.add_argument("--frames", type=int, default=0, help="override the number of frames per step")
    ap.add_argument("--conv-impl", default="auto", choices=["auto", "tcgen05", "direct"])
    ap.add_argument("--micro-batch", type=int, default=0)
    ap.add_argument("--weights", default="lc", choices=["lc", "st"],
                    help="synthetic weight set: lc = random He-normal net (smooth p-map, ~29 %% of the pixels above the "
                         "threshold), st = surrogate for trained weights (sharp p-map peaks, a few %% above the threshold)")
    ap.add_argument("--fusion", default="auto", choices=["auto", "none", "all", "head", "pairs1"])
    ap.add_argument("--stem", default="auto", choices=["auto", "tensor", "cuda"],
                    help="K1 kernel: SMLM_STEM_AUTO / TENSOR (conv_chain.cu STEM variant) / CUDA_CORES (stem.cu)")
    ap.add_argument("--tile", type=int, default=-1, help="override the config's tile size (0: whole frames)")
    ap.add_argument("--tile-merge", default="auto", choices=["auto", "none", "row"],
                    help="row: one window per tile row (SMLM_TILE_MERGE_ROW); auto = row for a tiled config "
                         "(cfg 3: 408 vs 325 frames/s, profiles/bench_r2.md)")
    ap.add_argument("--precision", default="", choices=["", "bf16", "fp16"],
                    help="activation storage type of the variants study (SURVEY.md 8(f)-4); default: the config's")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="default cfg-1 run only: do not append the short runs of cfgs 2, 3, 4 and --net dloc")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank localises the config's full stack (replicas); "
                         "strong = the stack is sharded by frame range (shard_frames)")
    ap.add_argument("--disk", default="", help="also time smlm_localize_ring from a frame file written to this directory")
    ap.add_argument("--selftest-spawn", action="store_true",
                    help="CPU only: exercise the --gpus N spawn path, the frame sharding and the max-over-ranks "
                         "reduction over gloo with synthetic per-rank timings")
    args = ap.parse_args(argv)
    if args.steps <= 0:
        args.steps = 5 if args.net == "dloc" else {2: 5, 3: 3, 4: 4}.get(args.config, 40)
    cfg = get_config(args.config)
    if args.tile >= 0 or args.precision:
        import dataclasses
        if args.tile >= 0:
            cfg = dataclasses.replace(cfg, tile=args.tile)
        if args.precision:
            cfg = dataclasses.replace(cfg, net=dataclasses.replace(cfg.net, precision=args.precision))
    if args.net == "dloc":
        args.warmup = max(args.warmup, 3)
        return run_dloc(args, cfg)
    if args.impl == "reference":
        return run_reference(args, cfg)
    args.warmup = max(args.warmup, 3)
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        return spawn_ranks(args, sys.argv[1:] if argv is None else list(argv))
    if args.selftest_spawn:
        return selftest_spawn(args, cfg)

    import torch
    import paper_2410_02314_b200 as P

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")     # the communicator line (nranks) goes to stderr
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    n_frames = args.frames or cfg.frames.n_frames
    if world > 1 and args.scaling == "strong":          # frame-range sharding, no exchange step
        from paper_2410_02314_b200.replicas import shard_frames
        lo, hi = shard_frames(n_frames, rank, world)
        n_frames = hi - lo
    fs, frames = workload(cfg, n_frames)
    weights = make_weights(cfg, args.weights)
    H, W = frames.shape[1:]
    conv_impl = {"auto": P.CONV_AUTO, "tcgen05": P.CONV_TCGEN05, "direct": P.CONV_DIRECT}[args.conv_impl]
    tile_merge = args.tile_merge if args.tile_merge != "auto" else ("row" if cfg.tile else "none")
    desc = P.desc_from_spec(cfg.net, tile=cfg.tile, micro_batch=args.micro_batch, conv_impl=conv_impl,
                            writeback_frames=cfg.writeback_batch,
                            tile_merge={"none": P.TILE_MERGE_NONE, "row": P.TILE_MERGE_ROW}[tile_merge],
                            stem_impl={"auto": P.STEM_AUTO, "tensor": P.STEM_TENSOR, "cuda": P.STEM_CUDA_CORES}[args.stem],
                            fusion={"auto": P.FUSE_AUTO, "none": P.FUSE_NONE, "all": P.FUSE_ALL, "head": P.FUSE_HEAD, "pairs1": P.FUSE_PAIRS_1CTA}[args.fusion])
    loc = P.Localizer(desc, weights)
    cap = int(n_frames * max(4 * cfg.frames.emitters_per_frame, 1024))
    cap = min(cap, n_frames * ((H + 1) // 2) * ((W + 1) // 2))
    off_map = torch.from_numpy(fs.offset_map).cuda() if fs.offset_map is not None else None
    gain_map = torch.from_numpy(fs.gain_map).cuda() if fs.gain_map is not None else None
    cam = loc.camera(fs.pixel_size_nm, fs.offset, fs.gain, off_map, gain_map)
    frames_host = torch.from_numpy(frames).pin_memory()
    frames_dev = frames_host.cuda()
    out_dev = torch.zeros(cap * 32, dtype=torch.uint8, device="cuda")
    out_host = torch.zeros(cap * 32, dtype=torch.uint8).pin_memory()
    stream = torch.cuda.Stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(frames_t, out_t, steps, kernel_timing=False):
        loc.kernel_timing(kernel_timing)
        barrier()
        l0 = loc.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        counts = []
        with torch.cuda.stream(stream):
            e0.record(stream)
            for _ in range(steps):
                counts.append(loc.localize(frames_t, cam, cfg.threshold, out_t, cap, stream=stream))
            e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        st = loc.check()
        if st != P.OK:
            raise SystemExit(f"smlm_check: {st} {loc.last_error()}")
        kt = {k: loc.kernel_time_ms(k) for k in (P.KERNEL_STEM, P.KERNEL_CONV, P.KERNEL_CONV_PAIR, P.KERNEL_POST)} \
            if kernel_timing else None
        loc.kernel_timing(False)
        return ms, [int(c.value) for c in counts], loc.launch_count() - l0, kt

    # warm-up (device-resident and end-to-end paths): W steps each, then more device-resident
    # steps until ~1.5 s of GPU work has run, so that the power-cap governor has settled (a
    # process started on an idle GPU measured ~3 % low in its first second)
    sampler = ClockSampler(local)                      # (NVML initialised here, outside the timed region)
    ms_w = timed(frames_dev, out_dev, args.warmup)[0]
    timed(frames_host, out_host, args.warmup)
    per_step = max(ms_w / args.warmup, 1e-3)
    extra = int(min(200, max(0.0, 1500.0 - ms_w) / per_step))
    if extra > 0:
        timed(frames_dev, out_dev, extra)
        timed(frames_host, out_host, max(1, extra // 3))

    sampler.start()
    # the timed window (exactly --steps steps) runs REPEATS times per path; `value` / `e2e` come from
    # the median window, all windows are listed under "repeats" (run-to-run spread of the power governor)
    reps_dev = [timed(frames_dev, out_dev, args.steps) for _ in range(REPEATS)]
    reps_e2e = [timed(frames_host, out_host, args.steps) for _ in range(REPEATS)]
    ms, counts, launches, _ = sorted(reps_dev, key=lambda r: r[0])[REPEATS // 2]
    ms_e2e, counts_e2e, _, _ = sorted(reps_e2e, key=lambda r: r[0])[REPEATS // 2]
    # roofline pass: the same steps with every K2 launch bracketed by CUDA events on the
    # launching stream (the events serialise a little, so `value` is not taken from this pass)
    ms_rf, _, _, kt = timed(frames_dev, out_dev, args.steps, kernel_timing=True)
    single_ms, single_n = kt[P.KERNEL_CONV]          # launches of one trunk layer
    pair_ms, pair_n = kt[P.KERNEL_CONV_PAIR]         # launches of two trunk layers (conv_pair.cu)
    conv_ms, conv_n = single_ms + pair_ms, single_n + pair_n
    disk = None
    if args.disk:
        # the paper's storage -> GPU experiment: reader threads fill the pinned ring
        # from a raw frame file while earlier chunks are localised (smlm_localize_ring)
        os.makedirs(args.disk, exist_ok=True)
        path = os.path.join(args.disk, f"bench_frames_rank{rank}.u16")
        frames.tofile(path)
        chunk, slots, threads = 256, 4, 4
        with P.Ring(path, n_frames, H, W, chunk, n_slots=slots, n_threads=threads) as ring:
            loc.localize_ring(ring, cam, cfg.threshold, out_host, cap, stream=stream)    # warm-up (page cache)
            torch.cuda.synchronize()
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            disk_counts = []      # kept until the barrier: the library writes them asynchronously
            for _ in range(args.steps):
                disk_counts.append(loc.localize_ring(ring, cam, cfg.threshold, out_host, cap, stream=stream))
            e1.record(stream)
            barrier()
            ms_disk = e0.elapsed_time(e1)
            if loc.check() != P.OK or any(int(c.value) != int(disk_counts[0].value) for c in disk_counts):
                raise SystemExit(f"--disk: smlm_check {loc.check()} / counts differ between passes")
        os.remove(path)
        disk = {"value": n_frames * args.steps / (ms_disk * 1e-3), "unit": UNIT, "ms_per_step": ms_disk / args.steps,
                "file_bytes": int(frames.nbytes), "chunk_frames": chunk, "ring_slots": slots, "reader_threads": threads,
                "note": "file re-read from the OS page cache after the warm-up pass"}
    sampler.stop_flag.set()
    sampler.join(timeout=2)

    from paper_2410_02314_b200.replicas import job_throughput
    # replicas only: units summed over ranks / slowest rank's device time
    value, ms_max = job_throughput(n_frames * args.steps, ms, dist, "cuda")
    e2e_value, ms_e2e_max = job_throughput(n_frames * args.steps, ms_e2e, dist, "cuda")
    emitters = sum(counts)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peaks, peak_kind = load_peaks()
    C, L = cfg.net.channels, cfg.net.n_layers
    # views of a full-size launch (api.cu auto_micro_batch: <= 128, <= 1.5 GB per activation buffer)
    if args.micro_batch:
        loc_views_per_launch = args.micro_batch
    elif cfg.tile and tile_merge == "none":   # the largest launch set: all interior tiles of the chunk's frames
        ext = cfg.tile + 2 * (cfg.net.radius + 1)
        mb = int(min(128, max(1, (1536 << 20) // (ext * ext * C * 2))))
        inner = max(1, (-(-H // cfg.tile) - 2)) * max(1, (-(-W // cfg.tile) - 2))
        loc_views_per_launch = max(1, min(mb // inner, n_frames)) * inner
    elif cfg.tile:                            # row-merged tiles: windows of (tile + 2 halo) rows x the frame width
        ext = cfg.tile + 2 * (cfg.net.radius + 1)
        mb = int(min(128, max(1, (1536 << 20) // (ext * W * C * 2))))
        inner = max(1, (-(-H // cfg.tile) - 2))
        loc_views_per_launch = max(1, min(mb // inner, n_frames)) * inner
    else:
        loc_views_per_launch = int(min(128, max(1, (1536 << 20) // (H * W * C * 2)), n_frames))
    # dominant kernel: the dilated 3x3 conv (K2), one layer per launch (conv_umma_kernel) or two
    # (conv_pair_kernel).  Algorithmic work = 18 C^2 FLOP per pixel per layer;
    # algorithmic bytes of a launch = 2C B/px in + 2C B/px out, whatever the number of layers it runs.
    flop_total = 18.0 * C * C * H * W * n_frames * L * args.steps
    roofline = None
    if conv_n > 0 and conv_ms > 0:  # tiled configs: algorithmic (whole-frame) FLOPs, halo recompute not counted
        achieved = flop_total / (conv_ms * 1e-3) / 1e12
        peak = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
        bound = "tensor"
        if cfg.net.precision not in ("bf16", "fp16") or args.conv_impl == "direct":
            bound = "alu"
        # the launches of the step split by kernel: layers = single_n + 2 pair_n
        layers_run = single_n + 2 * pair_n
        dominant_pair = pair_ms >= single_ms
        dom_ms, dom_n, dom_layers = (pair_ms, pair_n, 2) if dominant_pair else (single_ms, single_n, 1)
        dom_flop = flop_total * (dom_layers * dom_n) / layers_run
        alg_bytes_per_launch = 4.0 * C * H * W * n_frames * args.steps * L / layers_run
        # DRAM traffic per launch: dram__bytes_read.sum + dram__bytes_write.sum of the dominant
        # kernel in this launch shape, from the tracked ncu --set full record
        # (profiles/traffic_r2.json: per-kernel means of one `ncu --set full` capture, named there); null when no capture of this (workload, views per launch) exists.
        traffic, traffic_note = lookup_traffic(cfg, C, loc_views_per_launch, bound, dominant_pair, args.fusion)
        roofline = {"bound": bound,
                    "kernel": "conv3x3_dilated x2, layers (d, 2d) fused (conv_pair_kernel)" if dominant_pair
                              else "conv3x3_dilated (conv_umma_kernel)",
                    "achieved": dom_flop / (dom_ms * 1e-3) / 1e12, "peak": peak,
                    "unit": "TFLOP/s", "frac": dom_flop / (dom_ms * 1e-3) / 1e12 / peak,
                    "traffic": traffic, "traffic_source": traffic_note,
                    "algorithmic_bytes_per_launch": alg_bytes_per_launch,
                    "hbm_GBs_algorithmic": alg_bytes_per_launch * dom_n / (dom_ms * 1e-3) / 1e9,
                    "hbm_frac_algorithmic": alg_bytes_per_launch * dom_n / (dom_ms * 1e-3) / 1e9
                                            / float(peaks["hbm_gbs"]),
                    "peak_source": f"{peak_kind} bf16_tflops_sustained (kernel timed inside a long step)",
                    "frac_of_burst": dom_flop / (dom_ms * 1e-3) / 1e12 / float(peaks["bf16_tflops"]),
                    "launches": dom_n, "avg_launch_ms": dom_ms / dom_n, "layers_per_launch": dom_layers,
                    "share_of_step": dom_ms / ms_rf,
                    "all_trunk_launches": {"achieved": achieved, "frac": achieved / peak,
                                           "frac_of_burst": achieved / float(peaks["bf16_tflops"]),
                                           "single_layer_launches": single_n, "pair_launches": pair_n,
                                           "share_of_step": conv_ms / ms_rf}}
    # K1 / K3: bytes moved per launch / CUDA-event time, against the
    # measured HBM copy bandwidth.  K1 is a pure WRITE stream (2 B in, 2C B out per pixel); a
    # plain fill of device memory, measured here, is its real roof (profiles/stem_r2.md).
    fill = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    write_modes = {}
    for mode, label in ((0, "cudaMemsetAsync"), (1, "st.global.v4 kernel (smlm_debug_fill)")):
        best = 1e9
        for _ in range(10):
            f0.record()
            P.debug_fill(fill, mode)
            f1.record()
            torch.cuda.synchronize()
            best = min(best, f0.elapsed_time(f1))
        write_modes[label] = fill.numel() / (best * 1e-3) / 1e9
    write_src, write_gbs = max(write_modes.items(), key=lambda kv: kv[1])
    del fill
    io_kernels = {}
    if kt is not None:
        px = float(H) * W * n_frames * args.steps
        emit_bytes = 32.0 * sum(counts)
        for name, kind, nbytes in (("stem (K1)", P.KERNEL_STEM, px * (2 + 2 * C)),
                                   ("heads+post (K3)", P.KERNEL_POST, px * 4 + emit_bytes)):
            k_ms, k_n = kt[kind]
            if k_n > 0 and k_ms > 0:
                gbs = nbytes / (k_ms * 1e-3) / 1e9
                io_kernels[name] = {"achieved_GBs": gbs, "frac_of_hbm": gbs / float(peaks["hbm_gbs"]),
                                    "launches": k_n, "avg_launch_ms": k_ms / k_n,
                                    "share_of_step": k_ms / ms_rf}
                if kind == P.KERNEL_STEM:
                    io_kernels[name]["frac_of_write_stream_peak"] = gbs / write_gbs
                    io_kernels[name]["write_stream_peak_GBs"] = write_gbs
                    io_kernels[name]["write_stream_peak_source"] = f"{write_src}, 1 GiB, best of 10, this run"
                    io_kernels[name]["write_only_GBs"] = write_modes
    cpu = None
    if not args.no_cpu_baseline:
        # bounded sample: about 2e12 FLOP of oracle work (10-15 s on 16 host cores)
        ns = max(1, min(len(fs.frames), int(2e12 / (cfg.net.flop_per_px() * H * W))))
        fps, eps, cores, dt = oracle_sample(cfg, fs, weights, ns)
        cpu = {"value": fps, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {ns} frame(s) of {cfg.name}, {dt:.1f} s", "emitters_per_s": eps}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": args.scaling, "vs_baseline": None,
        "dtype": {"bf16": "bf16", "fp16": "f16"}.get(cfg.net.precision, "f32"), "data": "synthetic",
        "config": {"workload": cfg.name, "frames_per_step": n_frames, "H": H, "W": W, "channels": C,
                   "layers": L, "head_channels": cfg.net.head_channels, "tile": cfg.tile, "tile_merge": tile_merge,
                   "precision": cfg.net.precision, "weights": args.weights,
                   "distinct_frames": int(len(fs.frames)), "conv_impl": args.conv_impl, "fusion": args.fusion, "stem": args.stem,
                   "l2": "inputs larger than L2 (u16 stack + activation stream per step > 126 MB)",
                   "parallelism": f"replicas x{world}"},
        "emitters_per_s": world * emitters / (ms_max * 1e-3),
        "emitters_per_frame": emitters / (n_frames * args.steps),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(frames.nbytes),
                "d2h_bytes_per_step": int(counts_e2e[-1] * 32 + 8), "ms_per_step": ms_e2e_max / args.steps,
                "exposed_copy_ms_per_step": (ms_e2e_max - ms_max) / args.steps},
        "gpu_launches": launches,
        "clocks": sampler.summary(),
        "roofline": roofline,
        "io_kernels": io_kernels,
        "cpu_baseline": cpu,
        "from_disk": disk,
        "tensor_frac_whole_step": (cfg.net.flop_per_px() * H * W * n_frames * args.steps / (ms_max * 1e-3) / 1e12)
                                  / float(peaks["bf16_tflops"]),
        "repeats": {"windows": REPEATS, "steps_per_window": args.steps, "reported": "median window",
                    "value": sorted(world * n_frames * args.steps / (r[0] * 1e-3) for r in reps_dev),
                    "e2e": sorted(world * n_frames * args.steps / (r[0] * 1e-3) for r in reps_e2e),
                    "note": "this rank's windows x world size" if world > 1 else "frames/s of each window, ascending"},
    }
    if world == 1 and args.config == 1 and not args.frames and not args.no_other_configs and not args.disk:
        line["other_configs"] = other_configs(args)
    print(json.dumps(line), flush=True)
    loc.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
