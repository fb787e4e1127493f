"""Turns profiler output into the text records kept under profiles/ (nothing here runs on the
hot path; bench.py only READS profiles/traffic_r2.json).

    # opcode histogram of every kernel of the built library (cuobjdump -sass), markdown
    python -m paper_2410_02314_b200.profile_tools sass > profiles/sass_r2.md

    # DRAM traffic per launch from an `ncu --set full` capture exported with
    #   ncu -i capture.ncu-rep --page raw --csv > raw.csv
    python -m paper_2410_02314_b200.profile_tools traffic raw.csv --workload cfg1 --views 64 \
        --dilations 1,2,4,8 --merge profiles/traffic_r2.json

    # per-kernel totals of an `ncu --metrics gpu__time_duration.sum --csv` launch list, markdown
    python -m paper_2410_02314_b200.profile_tools launches launches.csv

    # device timeline of ONE end-to-end step (pinned frames in, pinned list out) from CUPTI via
    # torch.profiler: every H2D copy and kernel with start / end, and how much of the copy time
    # runs under a kernel (needs a GPU; markdown)
    python -m paper_2410_02314_b200.profile_tools timeline --config 1 > profiles/timeline_r2.md
"""
from __future__ import annotations

import argparse
import collections
import csv
import io
import json
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libsmlm_b200.so")

# mnemonics that prove the Blackwell paths (B200_PROFILING.md): tcgen05.mma / ld / st / commit,
# bulk (TMA) copies, mbarrier waits, packed fp32 FMA
KEY_OPS = ("UTCHMMA", "UTCQMMA", "UTCOMMA", "LDTM", "STTM", "UTCBAR", "UBLKCP", "UTMALDG", "SYNCS", "FFMA2",
           "FFMA", "HMMA", "LDS", "STS", "LDG", "STG", "ATOMS", "ATOMG", "RED", "BAR", "MUFU")


def demangle(name: str) -> str:
    if not name.startswith("_Z"):
        return name
    try:
        return subprocess.run(["c++filt", name], capture_output=True, text=True, check=True).stdout.strip()
    except (OSError, subprocess.CalledProcessError):
        return name


def short_name(name: str) -> str:
    """`conv_umma_kernel<48,HEAD,-,bf16>` style names from a mangled symbol or ncu's demangled one."""
    name = demangle(name)
    name = re.sub(r"^void\s+", "", name)
    for junk in ("smlm::", "(anonymous namespace)::", "<unnamed>::", "unnamed>::"):
        name = name.replace(junk, "")
    t = lambda v: v in ("1", "true")
    m = re.match(r"conv_umma_kernel<(\d+),\s*(?:\(bool\))?(\w+),\s*(?:\(bool\))?(\w+)(?:,\s*(?:\(bool\))?(\w+))?>", name)
    if m:
        return (f"conv_umma_kernel<{m.group(1)},{'HEAD' if t(m.group(2)) else '-'},"
                f"{'STEM' if t(m.group(3)) else '-'}" + (",f16" if m.group(4) and t(m.group(4)) else "") + ">")
    m = re.match(r"conv_pair_kernel<(\d+),\s*(?:\(bool\))?(\w+),\s*(?:\(bool\))?(\w+),\s*(?:\(bool\))?(\w+)>", name)
    if m:
        return (f"conv_pair_kernel<{m.group(1)},{'HEAD' if t(m.group(2)) else '-'},{'f16' if t(m.group(3)) else '-'},"
                f"{'cg2' if t(m.group(4)) else 'cg1'}>")
    m = re.match(r"conv_chain_kernel<(\d+),\s*(?:\(bool\))?(\w+),\s*(?:\(int\))?(\d+),\s*(?:\(bool\))?(\w+)>", name)
    if m:
        return (f"conv_chain_kernel<{m.group(1)},{'f16' if t(m.group(2)) else '-'},{m.group(3)},"
                f"{'STEM' if t(m.group(4)) else '-'}>")
    m = re.match(r"([\w:]+)(<.*?>)?\(", name)
    if m:
        return m.group(1) + (m.group(2) or "").replace("__nv_bfloat16", "bf16").replace("__half", "f16") \
            .replace("float", "f32").replace(" ", "")
    return name[:60]


def cmd_sass(args):
    out = subprocess.run(["cuobjdump", "-sass", args.lib], capture_output=True, text=True, check=True).stdout
    kernels = collections.OrderedDict()
    cur = None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = kernels.setdefault(short_name(m.group(1)), collections.Counter())
            continue
        m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", line)
        if m and cur is not None:
            cur[m.group(1)] += 1
    print("# SASS opcode histogram of libsmlm_b200.so (sm_100a)\n")
    print("Command: `python -m paper_2410_02314_b200.profile_tools sass` (runs `cuobjdump -sass` on the in-tree "
          "library built by `paper_2410_02314_b200/build.py`).\n")
    print("UTCHMMA = tcgen05.mma kind::f16, LDTM / STTM = tcgen05.ld / st, UTCBAR = tcgen05.commit, UBLKCP = "
          "cp.async.bulk (1-D TMA), SYNCS = mbarrier, FFMA2 = fma.rn.f32x2.\n")
    ops = [o for o in KEY_OPS if any(c[o] for c in kernels.values())]
    print("| kernel | instr | " + " | ".join(ops) + " |")
    print("|---|---|" + "---|" * len(ops))
    for name, c in kernels.items():
        if args.filter and not re.search(args.filter, name):
            continue
        print(f"| `{name}` | {sum(c.values())} | " + " | ".join(str(c[o]) for o in ops) + " |")
    return 0


def read_ncu_raw(path):
    """`ncu --page raw --csv`: one row per launch, header row + units row."""
    with open(path, "r", encoding="utf-8", errors="replace") as fh:
        text = fh.read()
    start = text.find('"ID"')
    rows = list(csv.reader(io.StringIO(text[start:])))
    hdr = rows[0]
    units = rows[1]
    body = [dict(zip(hdr, r)) for r in rows[2:] if len(r) == len(hdr)]
    return hdr, dict(zip(hdr, units)), body


def to_bytes(val: str, unit: str) -> float:
    v = float(val.replace(",", ""))
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    return v * scale.get(unit, 1.0)


def to_ns(val: str, unit: str) -> float:
    v = float(val.replace(",", ""))
    return v * {"ns": 1.0, "us": 1e3, "usecond": 1e3, "ms": 1e6, "msecond": 1e6, "s": 1e9, "second": 1e9,
                "nsecond": 1.0}.get(unit, 1.0)


def cmd_traffic(args):
    _, units, body = read_ncu_raw(args.csv)
    dil = [int(x) for x in args.dilations.split(",")] if args.dilations else []
    entries = []
    per_kernel_idx = collections.Counter()
    for r in body:
        name = short_name(r["Kernel Name"])
        i = per_kernel_idx[name]
        per_kernel_idx[name] += 1
        rd = to_bytes(r["dram__bytes_read.sum"], units["dram__bytes_read.sum"])
        wr = to_bytes(r["dram__bytes_write.sum"], units["dram__bytes_write.sum"])
        e = {"kernel": name, "launch": int(r["ID"]), "grid": r.get("Grid Size", ""), "block": r.get("Block Size", ""),
             "dram_read_bytes": rd, "dram_write_bytes": wr, "dram_bytes": rd + wr,
             "duration_us": to_ns(r["gpu__time_duration.sum"], units["gpu__time_duration.sum"]) / 1e3}
        for key, label in (("sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_elapsed", "tensor_pipe_pct_elapsed"),
                           ("sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "tensor_pipe_pct_active"),
                           ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue_active_pct"),
                           ("dram__throughput.avg.pct_of_peak_sustained_elapsed", "dram_pct"),
                           ("lts__t_sector_hit_rate.pct", "l2_hit_pct"),
                           ("sm__throughput.avg.pct_of_peak_sustained_elapsed", "sm_pct")):
            if key in r and r[key] not in ("", "n/a"):
                try:
                    e[label] = float(r[key].replace(",", ""))
                except ValueError:
                    pass
        entries.append(e)
    # conv launches come in layer order; label their dilation when the cycle is given
    if dil:
        k = 0
        for e in entries:
            if e["kernel"].startswith("conv_umma_kernel"):
                e["dilation"] = dil[k % len(dil)]
                k += 1
            elif e["kernel"].startswith("conv_pair_kernel"):   # two layers per launch
                e["dilation"] = [dil[k % len(dil)], dil[(k + 1) % len(dil)]]
                k += 2
    record = {"workload": args.workload, "views_per_launch": args.views, "source": args.source or args.csv,
              "launches": entries}
    by = collections.defaultdict(list)
    for e in entries:
        by[e["kernel"]].append(e)
    record["per_kernel_mean"] = {
        k: {"n": len(v), "dram_bytes": sum(x["dram_bytes"] for x in v) / len(v),
            "dram_read_bytes": sum(x["dram_read_bytes"] for x in v) / len(v),
            "dram_write_bytes": sum(x["dram_write_bytes"] for x in v) / len(v),
            "duration_us": sum(x["duration_us"] for x in v) / len(v)} for k, v in by.items()}
    if args.merge:
        doc = {"written_by": "python -m paper_2410_02314_b200.profile_tools traffic", "captures": {}}
        if os.path.exists(args.merge):
            with open(args.merge, "r", encoding="utf-8") as fh:
                doc = json.load(fh)
        doc["captures"][f"{args.workload}/views{args.views}" + (f"/{args.tag}" if args.tag else "")] = record
        with open(args.merge, "w", encoding="utf-8") as fh:
            json.dump(doc, fh, indent=1, sort_keys=True)
    else:
        json.dump(record, sys.stdout, indent=1, sort_keys=True)
    return 0


def cmd_launches(args):
    with open(args.csv, "r", encoding="utf-8", errors="replace") as fh:
        text = fh.read()
    rows = list(csv.DictReader(io.StringIO(text[text.find('"ID"'):])))
    tot = collections.OrderedDict()
    for r in rows:
        if r.get("Metric Name") != "gpu__time_duration.sum":
            continue
        n = short_name(r["Kernel Name"])
        t = tot.setdefault(n, [0, 0.0, r["Grid Size"], r["Block Size"]])
        t[0] += 1
        t[1] += to_ns(r["Metric Value"], r["Metric Unit"]) / 1e3
    all_us = sum(t[1] for t in tot.values())
    print("| kernel | launches | total us | mean us | share | grid | block |")
    print("|---|---|---|---|---|---|---|")
    for n, (k, us, grid, block) in tot.items():
        print(f"| `{n}` | {k} | {us:.1f} | {us / k:.1f} | {100 * us / all_us:.1f} % | {grid} | {block} |")
    return 0


def cmd_timeline(args):
    """One smlm_localize call with the frames in pinned host memory and the list in pinned host
    memory, traced by CUPTI (torch.profiler).  Not a timing run: the profiler adds overhead."""
    import numpy as np
    import torch
    from torch.profiler import ProfilerActivity, profile
    root = os.path.dirname(HERE)
    if root not in sys.path:
        sys.path.insert(0, root)
    import paper_2410_02314_b200 as P
    from smlm_synth import get_config, make_frames, make_weights
    cfg = get_config(args.config)
    n = args.frames or cfg.frames.n_frames
    fs = make_frames(cfg, min(64, n))
    frames = np.ascontiguousarray(np.concatenate([fs.frames] * (-(-n // len(fs.frames))))[:n])
    loc = P.Localizer(P.desc_from_spec(cfg.net, tile=cfg.tile, writeback_frames=cfg.writeback_batch), make_weights(cfg))
    H, W = frames.shape[1:]
    cap = int(min(n * ((H + 1) // 2) * ((W + 1) // 2), n * max(4 * cfg.frames.emitters_per_frame, 1024)))
    om = torch.from_numpy(fs.offset_map).cuda() if fs.offset_map is not None else None
    gm = torch.from_numpy(fs.gain_map).cuda() if fs.gain_map is not None else None
    cam = loc.camera(fs.pixel_size_nm, fs.offset, fs.gain, om, gm)
    fh = torch.from_numpy(frames).pin_memory()
    oh = torch.zeros(cap * 32, dtype=torch.uint8).pin_memory()
    st = torch.cuda.Stream()
    for _ in range(3):
        loc.localize(fh, cam, cfg.threshold, oh, cap, stream=st)
    torch.cuda.synchronize()
    with profile(activities=[ProfilerActivity.CUDA]) as prof:
        loc.localize(fh, cam, cfg.threshold, oh, cap, stream=st)
        torch.cuda.synchronize()
    ev = sorted((e.time_range.start, e.time_range.end, short_name(e.name) if "smlm" in e.name else e.name)
                for e in prof.events() if e.device_type == torch.autograd.DeviceType.CUDA)
    t0 = ev[0][0]
    ev = [(a - t0, b - t0, nm) for a, b, nm in ev]
    copies = [(a, b) for a, b, nm in ev if nm.startswith("Memcpy HtoD")]
    kernels = sorted((a, b) for a, b, nm in ev if not nm.startswith("Mem"))
    merged = []                      # union of the kernel intervals
    for a, b in kernels:
        if merged and a <= merged[-1][1]:
            merged[-1][1] = max(merged[-1][1], b)
        else:
            merged.append([a, b])
    def under(a, b):
        return sum(max(0.0, min(b, y) - max(a, x)) for x, y in merged)
    copy_us = sum(b - a for a, b in copies)
    hidden = sum(under(a, b) for a, b in copies)
    end = max(b for _, b, _ in ev)
    busy = sum(y - x for x, y in merged)
    print(f"# Device timeline of one end-to-end step (cfg {args.config}, {n} frames), round 2\n")
    print(f"Command: `python -m paper_2410_02314_b200.profile_tools timeline --config {args.config}"
          + (f" --frames {args.frames}" if args.frames else "") + "` (CUPTI activity records through `torch.profiler`; one "
          "`smlm_localize` call with the frames in pinned host memory and the emitter list in pinned host memory, after "
          "three warm-up calls).  The profiler adds overhead: this is a picture of the overlap, not a timing.\n")
    print(f"* step on the device: {end / 1e3:.2f} ms; kernels busy {busy / 1e3:.2f} ms ({100 * busy / end:.1f} %)")
    print(f"* H2D copies: {len(copies)}, {copy_us / 1e3:.2f} ms in total, {100 * hidden / max(copy_us, 1e-9):.1f} % of it under a "
          f"running kernel; first kernel starts at {kernels[0][0]:.0f} us")
    print(f"* consecutive trunk launches overlap by programmatic dependent launch: the next kernel's start precedes "
          f"the previous kernel's end\n")
    print("| start us | end us | activity |")
    print("|---|---|---|")
    for a, b, nm in ev[:args.rows]:
        print(f"| {a:.1f} | {b:.1f} | `{nm[:90]}` |")
    if len(ev) > args.rows:
        print(f"| ... | ... | {len(ev) - args.rows} more activities |")
    loc.close()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    sub = ap.add_subparsers(dest="cmd", required=True)
    s = sub.add_parser("sass")
    s.add_argument("--lib", default=LIB)
    s.add_argument("--filter", default="")
    s.set_defaults(fn=cmd_sass)
    t = sub.add_parser("traffic")
    t.add_argument("csv")
    t.add_argument("--workload", required=True)
    t.add_argument("--views", type=int, required=True)
    t.add_argument("--dilations", default="")
    t.add_argument("--tag", default="")
    t.add_argument("--source", default="")
    t.add_argument("--merge", default="")
    t.set_defaults(fn=cmd_traffic)
    l = sub.add_parser("launches")
    l.add_argument("csv")
    l.set_defaults(fn=cmd_launches)
    tl = sub.add_parser("timeline")
    tl.add_argument("--config", type=int, default=1)
    tl.add_argument("--frames", type=int, default=0)
    tl.add_argument("--rows", type=int, default=48)
    tl.set_defaults(fn=cmd_timeline)
    args = ap.parse_args(argv)
    return args.fn(args)


if __name__ == "__main__":
    sys.exit(main())
