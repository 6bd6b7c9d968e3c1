"""Host logic of bench.py's multi-rank paths on CPU (gloo, world size 2): the two sharding plans, the max-over-ranks
timing, the gather of the per-rank event lists of the template-sharded mode, and the self-launch of N ranks."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

TRIG = np.dtype([("template_id", np.int32), ("sample", np.int32), ("rho", np.float32), ("chisq", np.float32)])


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    weak = bench.shard_plan(world, rank, 1024)
    strong = bench.shard_plan(world, rank, 1023, "templates")
    ms = bench.reduce_max_ms(10.0 + 5.0 * rank, dist)
    # template-sharded mode: rank r found r + 2 events in its range of template ids
    mine = np.zeros(rank + 2, dtype=TRIG)
    mine["template_id"] = strong[1] + np.arange(rank + 2)
    mine["sample"] = 100 * rank + np.arange(rank + 2)
    mine["rho"] = 6.5 + rank
    allt = bench.gather_triggers(mine, dist)
    q.put((rank, weak, strong, ms, allt.tobytes()))
    dist.barrier()
    dist.destroy_process_group()


def test_world2_gloo_sharding_timing_and_gather():
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
    # weak scaling: each rank owns the whole bank against its own segment (distinct seeds)
    assert [r[1] for r in rows] == [(0, 0, 1024), (1, 0, 1024)]
    # strong scaling: one segment (seed offset 0), contiguous template ranges that tile the bank
    assert [r[2] for r in rows] == [(0, 0, 512), (0, 512, 511)]
    # every rank sees the same, maximal, time
    assert all(r[3] == 15.0 for r in rows)
    # both ranks hold the same gathered list: rank 0's 2 events, then rank 1's 3, template ids ascending
    a = np.frombuffer(rows[0][4], dtype=TRIG)
    assert rows[0][4] == rows[1][4] and len(a) == 5
    assert list(a["template_id"]) == [0, 1, 512, 513, 514] and list(a["sample"]) == [0, 1, 100, 101, 102]


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max_ms(3.5) == 3.5
    assert bench.shard_plan(1, 0, 7) == (0, 0, 7)
    assert bench.shard_plan(1, 0, 7, "templates") == (0, 0, 7)
    t = np.zeros(3, dtype=TRIG)
    assert bench.gather_triggers(t) is t
    for world in (2, 3, 8):
        plans = [bench.shard_plan(world, r, 1024, "templates") for r in range(world)]
        assert plans[0][1] == 0 and sum(p[2] for p in plans) == 1024
        assert all(plans[r][1] + plans[r][2] == plans[r + 1][1] for r in range(world - 1))
    peak, src = bench.measured_peak()
    assert peak > 1000 and ("measured" in src or "fallback" in src)


def test_gpus_n_without_a_launcher_starts_n_ranks(monkeypatch):
    # `python bench.py --gpus 2` must start two ranks itself (torchrun, 127.0.0.1), not run one process that claims two
    sys.path.insert(0, ROOT)
    import bench
    seen = {}
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "2", "--steps", "1"])
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    assert bench.main() == 0
    cmd = seen["cmd"]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=2" in cmd and "127.0.0.1" in cmd
    assert cmd[-4:] == ["--gpus", "2", "--steps", "1"] and cmd[-5].endswith("bench.py")


def test_world_size_must_match_gpus(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("WORLD_SIZE", "2")
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4"])
    with pytest.raises(AssertionError):
        bench.main()
