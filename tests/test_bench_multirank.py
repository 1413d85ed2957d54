"""N > 1 path of bench.py on CPU (gloo, world_size 2): the path is "replicas only" -- every rank builds
its own Sigma and the only collectives are the timing barrier and the max over ranks of the rank-local time."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_ms = 100.0 + 25.0 * rank                      # rank 1 is the slow replica
    ms = bench.max_over_ranks(local_ms, world, "cpu")
    dist.barrier()
    out[rank] = (ms, bench.whole_job_value(1e12, world, ms))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    world, port = 2, 29500 + (os.getpid() % 2000)
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    assert set(out.keys()) == {0, 1}
    for rank in range(world):
        ms, value = out[rank]
        assert ms == 125.0                               # the max, on every rank
        assert value == pytest.approx(2 * 1e12 / 0.125 / 1e12)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.whole_job_value(2e12, 1, 1000.0) == pytest.approx(2.0)


def test_reference_arm_ranks_other_than_zero_exit_without_work(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    args = type("A", (), {"workload": "tiny", "steps": 1, "warmup": 0, "gpus": 2, "ref_poles": 0})()
    assert bench.run_reference(args) == 0
