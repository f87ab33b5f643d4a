"""N > 1 is "replicas only": the path has no exchange step, so the only
multi-rank logic is bench.py's timing reduction (max over ranks) and the whole-job value.
Covered here with two gloo ranks on the CPU."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    tmax = bench.max_over_ranks(ms, world, "cpu")
    out[rank] = (tmax, bench.job_value(1000, 4, world, tmax))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world2():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    tmax, value = res[0]
    assert tmax == 15.0
    assert value == pytest.approx(2 * 1000 * 4 / 15e-3 / 1e6)


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.job_value(10 ** 6, 2, 1, 1.0) == pytest.approx(2000.0)
