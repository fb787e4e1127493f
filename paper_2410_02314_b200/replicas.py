"""Multi-GPU = independent replicas (BASELINE.json: one GPU, no sharding,
no collectives on the data path).  Frames are independent, so rank r of N localises a
contiguous range of the stack on its own GPU; the only communication is bookkeeping done by
the harness: a barrier around the timed region and a MAX over ranks of the device time.
"""
from __future__ import annotations

from typing import Tuple


def shard_frames(n_frames: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous range [lo, hi) of rank `rank`; sizes differ by at most one frame."""
    if world < 1 or not 0 <= rank < world or n_frames < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_frames, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def job_throughput(units_local: float, ms_local: float, dist=None, device=None) -> Tuple[float, float]:
    """(whole-job units/s, max-over-ranks ms): units summed over ranks / slowest rank's time."""
    import torch
    t = torch.tensor([float(ms_local), float(units_local)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        mx = t[:1].clone()
        sm = t[1:].clone()
        dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        dist.all_reduce(sm, op=dist.ReduceOp.SUM)
        ms, units = float(mx.item()), float(sm.item())
    else:
        ms, units = float(t[0].item()), float(t[1].item())
    return (units / (ms * 1e-3) if ms > 0 else 0.0), ms
