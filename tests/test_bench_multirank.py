"""The N > 1 path of bench.py (independent replicas, one per rank) on CPU: two gloo ranks check
the max-over-ranks timing and the whole-job aggregate that rank 0 prints."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
        ms = bench.max_over_ranks(ms_local, world, "cpu")
        dist.barrier()
        out[rank] = (ms, bench.whole_job_value(2_469_600, world, 100, ms))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_aggregate():
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0                 # the slowest rank sets the job's time
    expected = 2 * 2_469_600 * 100 / 15e-3 / 1e9          # both replicas' DOFs over the max time
    assert res[0][1] == pytest.approx(expected) and res[1][1] == pytest.approx(expected)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.whole_job_value(1e9, 1, 10, 1000.0) == pytest.approx(10.0)
