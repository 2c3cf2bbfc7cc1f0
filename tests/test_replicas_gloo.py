"""N > 1 is "replicas only": no data-path collective, only the barrier and the max-over-ranks of the step
time.  This covers that host-side logic of bench.py with world_size = 2 on the gloo backend (CPU)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local = 0.010 if rank == 0 else 0.025                     # rank 1 is the slow replica
    t = bench.max_over_ranks(local, world, torch.device("cpu"))
    dist.barrier()
    out[rank] = (t, bench.job_throughput(1000, 7, world, t))
    dist.destroy_process_group()


def test_replicas_time_is_max_over_ranks_and_value_is_whole_job():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    t, v = res[0]
    assert t == 0.025
    assert v == 1000 * 7 * 2 / 0.025 / 1e6


def test_single_rank_needs_no_process_group():
    assert bench.max_over_ranks(0.5, 1, torch.device("cpu")) == 0.5
