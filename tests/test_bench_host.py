"""Host logic of bench.py's multi-rank path on CPU: sharding plan and max-over-ranks timing (gloo, world 2)."""
import os
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seed_off, first, count = bench.shard_plan(world, rank, 1024)
    ms = bench.reduce_max_ms(10.0 + 5.0 * rank, dist)
    q.put((rank, seed_off, first, count, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_world2_gloo_sharding_and_max_time():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 500)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    rows = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # weak scaling: each rank owns the whole bank against its own segment (distinct seeds), and every
    # rank sees the same, maximal, time
    assert [r[1] for r in rows] == [0, 1]
    assert all(r[2] == 0 and r[3] == 1024 for r in rows)
    assert all(r[4] == 15.0 for r in rows)


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max_ms(3.5) == 3.5
    assert bench.shard_plan(1, 0, 7) == (0, 0, 7)
    peak, src = bench.measured_peak()
    assert peak > 1000 and ("measured" in src or "fallback" in src)
