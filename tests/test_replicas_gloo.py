"""The N > 1 path of bench.py (replicas only): frame-range sharding and the max-over-ranks /
sum-over-ranks bookkeeping, on CPU with gloo, world_size 2."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2410_02314_b200.replicas import job_throughput, shard_frames


def test_shard_frames_partitions_exactly():
    for n in (0, 1, 7, 1000, 10001):
        for world in (1, 2, 3, 8):
            ranges = [shard_frames(n, r, world) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
            sizes = [hi - lo for lo, hi in ranges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_frames(10, 2, 2)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_frames(1001, rank, world)
    ms = 10.0 if rank == 0 else 25.0          # rank 1 is the slow one
    value, ms_max = job_throughput(hi - lo, ms, dist)
    out[rank] = (lo, hi, value, ms_max)
    dist.barrier()
    dist.destroy_process_group()


def test_job_throughput_is_sum_over_max_world2():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = mp.get_context("spawn").Manager().dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    (lo0, hi0, v0, m0), (lo1, hi1, v1, m1) = out[0], out[1]
    assert (lo0, hi0, lo1, hi1) == (0, 501, 501, 1001)
    assert m0 == m1 == 25.0
    assert v0 == v1 == pytest.approx(1001 / 0.025)


def test_job_throughput_single_process():
    v, ms = job_throughput(100, 50.0)
    assert ms == 50.0 and v == pytest.approx(2000.0)


@pytest.mark.parametrize("scaling,frames0,value", [("weak", 1000, 2000 / 11e-3), ("strong", 500, 1000 / 11e-3)])
def test_bench_spawns_its_own_ranks(scaling, frames0, value):
    """`python bench.py --gpus 2` without torchrun: bench.py starts the ranks itself
    (torch.multiprocessing.spawn), shards by frame range in the strong case and reports
    whole-job units / slowest rank's time.  Exercised on CPU over gloo with synthetic timings."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--selftest-spawn",
                          "--scaling", scaling], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == scaling and line["frames_rank0"] == frames0
    assert line["ms_max"] == pytest.approx(11.0) and line["value"] == pytest.approx(value)
