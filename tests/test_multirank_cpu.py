"""N > 1 host logic on CPU (gloo, world_size 2): the path is "replicas only", so the
only cross-rank step is the max-over-ranks of the timed region and the whole-job aggregate that rank 0 prints."""
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    per_rank_ms = 10.0 * (rank + 1)                      # rank 1 is the slow replica
    total = bench.max_over_ranks(per_rank_ms, world, "cpu")
    value = bench.whole_job_gcells_per_s(1_000_000, 5, world, total)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, total, value))


def test_max_over_ranks_and_whole_job_value_with_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, total, value in res:
        assert total == 20.0                              # the slowest rank's time, on every rank
        assert value == pytest.approx(2 * 1_000_000 * 5 / 20e-3 / 1e9)


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(7.5, 1, "cpu") == 7.5
    assert bench.whole_job_gcells_per_s(402653184, 10, 1, 115.9) == pytest.approx(34.74, rel=1e-3)


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""   # the other ranks exit 0 without work
