"""N > 1 host logic of bench.py ("replicas only") with world_size 2 on CPU (gloo):
the step time is the MAX over ranks and the whole-job rate counts every rank's cell updates."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 100.0 + 50.0 * rank                 # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world)
    dist.barrier()
    out[rank] = (ms, bench.whole_job_rate(1.0e9, 2, world, ms))
    dist.destroy_process_group()


def test_replicas_max_time_and_aggregate_rate():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 150.0                         # max over ranks, same on every rank
    assert res[0][1] == pytest.approx(2 * 1.0e9 * 2 / 0.150 / 1e9)  # both replicas' work / slowest time


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(12.5, 1) == 12.5
    assert bench.whole_job_rate(2.0e9, 1, 1, 1000.0) == pytest.approx(2.0)
