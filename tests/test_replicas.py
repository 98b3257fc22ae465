"""Multi-GPU path of bench.py on CPU: replicas only. Two gloo ranks
reduce their timings with the helper bench.py uses; the aggregate is total work / max time."""
import os
import socket
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
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [10.0, 14.0][rank]            # rank 1 is the slow replica
    e2e_s = [0.5, 0.4][rank]
    ms_all, e2e_all = bench.max_over_ranks([ms, e2e_s], world, torch.device("cpu"))
    out[rank] = (ms_all, e2e_all, bench.replicas_value(1000, 50, world, ms_all * 1e-3))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_aggregate_is_total_work_over_max_time():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        ms_all, e2e_all, value = res[rank]
        assert ms_all == 14.0 and e2e_all == 0.5
        assert value == pytest.approx(2 * 1000 * 50 / 14.0e-3 / 1e6)


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks([3.0, 1.0], 1, None) == [3.0, 1.0]
    assert bench.replicas_value(10, 10, 1, 1e-6) == pytest.approx(100.0)


def test_reference_arm_idles_on_other_ranks(monkeypatch):
    """Under torchrun only rank 0 runs the oracle; the others exit 0 without work."""
    import argparse
    import bench
    args = argparse.Namespace(workload="pipe", small=True, scheme=None, store="f64", steps=1, lattice="d3q15",
                              warmup=1, inner=2, ref_seconds=1.0, gpus=2)
    assert bench.run_reference(args, rank=1, world=2) == 0
