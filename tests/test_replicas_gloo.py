"""N > 1 is "replicas only": the only multi-rank logic is the MAX of the per-rank timings and the
aggregate throughput.  Covered here with world_size 2 on the gloo backend (CPU)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local = [10.0 + 5.0 * rank, 20.0 - 3.0 * rank]          # rank 1 is slower in the first timing, faster in the second
    t, e = bench.max_over_ranks(local, world, torch.device("cpu"))
    out[rank] = (t, e, bench.whole_job_value(1000, 4, world, t))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_value_world2():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29531, out), nprocs=2, join=True)
    for rank in (0, 1):
        t, e, v = out[rank]
        assert t == 15.0 and e == 20.0
        assert abs(v - 2 * 1000 * 4 / 15.0e-3) < 1e-6


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.5, 7.25], 1, torch.device("cpu")) == [3.5, 7.25]
    assert bench.whole_job_value(500, 10, 1, 2.0) == 500 * 10 / 2.0e-3


def test_gpus_flag_spawns_one_rank_per_gpu(monkeypatch):
    """`python bench.py --gpus N` outside torchrun launches N ranks itself (same line as the driver's torchrun call)."""
    sys.path.insert(0, ROOT)
    import bench
    seen = {}
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    assert bench.spawn_replicas(4, ["--gpus", "4", "--steps", "2"]) == 0
    cmd = seen["cmd"]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=4" in cmd and "127.0.0.1" in cmd
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and cmd[-5].endswith("bench.py")
