"""Host logic of bench.py for --gpus N > 1 (replicas only): max-over-ranks timing and
whole-job throughput, exercised with two gloo ranks on CPU."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r measured (10 + 5 r) ms for the resident loop and (30 + r) ms end to end
    ms, ms_e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 30.0 + rank], dist, torch.device("cpu"))
    out[rank] = (ms, ms_e2e, bench.whole_job_throughput(1000, 4, world, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_max_and_aggregate():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29533, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        ms, ms_e2e, val = res[r]
        assert ms == 15.0 and ms_e2e == 31.0            # the slowest rank defines the job
        assert val == pytest.approx(1000 * 3 * 4 * 2 / 15e-3 / 1e6)


def test_single_rank_passthrough():
    import bench
    assert bench.max_over_ranks([1.5, 2.5], None, torch.device("cpu")) == [1.5, 2.5]
    assert bench.whole_job_throughput(12_800_000, 10, 1, 120.0) == pytest.approx(3200.0)
