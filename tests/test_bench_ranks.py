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


def test_byte_formula_and_config_object():
    """bench.py's algorithmic bytes per cell-stage and the config object both arms print"""
    import argparse
    import bench
    import workloads as W
    wl = W.c4_jet(ni=20, nj=20, nk=20)
    b = bench.bytes_per_cell_stage(wl["params"], 0.25)
    # k_grad 12 doubles; eta 6 + 10 + 8 + 5 + 4; zeta 6 + 10 + 8 + 10; xi: + U, U^n, 1/J, sigma, Q_ref where sigma != 0, P_next
    assert b["grad"] == 96 and b["flux_eta"] == 264 and b["flux_zeta"] == 272
    assert b["flux_xi"] == pytest.approx(8 * (24 + 5 + 5 + 10 / 3 + 1 + (1 + 5 * 0.25) + 5 + 5 / 3 + 6))
    assert bench.bytes_per_cell_stage(wl["params"], None)["flux_xi"] == pytest.approx(b["flux_xi"] - 8 * 2.25)
    inv = bench.bytes_per_cell_stage(W.c1_vortex(n=16)["params"], None)
    assert inv["grad"] == 0 and inv["flux_eta"] == 8 * (5 + 3 + 5) and inv["metrics"] == 0
    mov = bench.bytes_per_cell_stage(W.c2_dynamic_freestream(n=16)["params"], None)
    assert mov["metrics"] > 0 and mov["flux_eta"] == inv["flux_eta"] + 8
    assert bench.sponge_fraction(wl) == pytest.approx((wl["sigma"] != 0).mean())
    cfg = bench.ref_config(argparse.Namespace(develop=None, warmup=5))
    assert cfg["workload"] == "c4_jet_320x200x200" and cfg["cells"] == 12_800_000 and cfg["dt"] == 2.0e-3
    assert "250 untimed steps" in cfg["state"] and "L2" in cfg["l2"]
