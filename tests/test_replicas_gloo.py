"""N > 1 path of bench.py on CPU: replicas only.  Two gloo ranks run the same host-side aggregation
the GPU bench uses (aggregate_over_ranks): whole-job time = MAX over ranks, whole-job work = SUM over ranks.  No data-path
collective exists to test: every rank solves its own copy."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" 10 + r ms for 100 + r iterations, 405 + 4 r launches, 5000 + 100 r iter/s end to end
    dist.barrier()
    res = bench.aggregate_over_ranks(dist, torch, 10.0 + rank, 100 + rank, 405 + 4 * rank, 5000.0 + 100 * rank, "cpu")
    out[rank] = res
    dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_replica_aggregation_world2():
    world = 2
    mgr = mp.get_context("spawn").Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    for rank in range(world):
        step_ms, total_it, launches, e2e = out[rank]
        assert step_ms == 11.0                 # max over ranks
        assert total_it == 201                 # sum of work
        assert launches == 405 + 409
        assert e2e == 10100.0
    # value = whole-job iterations / max time
    assert abs(out[0][1] / (out[0][0] * 1e-3) - 201 / 0.011) < 1e-6


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(None, torch, 3.5, 7, 33, 2.0, "cpu") == (3.5, 7, 33, 2.0)
