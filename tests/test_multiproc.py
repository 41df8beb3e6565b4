"""N > 1 path of bench.py (replicas only) with 2 gloo ranks on CPU:
the timing reduction is the max over ranks and the reported value is the whole-job aggregate."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = 2.0 + rank                       # rank 1 is the slow replica
    worst = bench.max_over_ranks(ms, world, device="cpu")
    dist.barrier()
    out[rank] = (worst, bench.whole_job_mlups(1_000_000, worst, world))
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_and_value_is_aggregate():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29617, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 3.0
    assert res[0][1] == pytest.approx(2 * 1_000_000 / 3.0 / 1e3)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.5, 1) == 1.5
    assert bench.whole_job_mlups(2_097_152, 0.1, 1) == pytest.approx(20971.52)
