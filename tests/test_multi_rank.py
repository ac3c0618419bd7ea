"""The N > 1 path of bench.py is "replicas only": the only inter-rank step is
the max-over-ranks timing and the whole-job throughput arithmetic.  World size 2, gloo, on CPU."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 * (rank + 1), dist, device="cpu")      # rank 0: 10 ms, rank 1: 20 ms
    value = bench.whole_job_value(rows_per_rank=1000, world=world, steps=4, ms=ms)
    out[rank] = (ms, value)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        ms, value = res[rank]
        assert ms == 20.0                                  # the slowest rank's time, on every rank
        assert value == 1000 * world * 4 / 20e-3           # all ranks' rows / that time


def test_seed_offsets_differ_per_rank():
    a = bench.build_workload("C1", "cpu", scale=100, seed_offset=0)
    b = bench.build_workload("C1", "cpu", scale=100, seed_offset=1)
    assert not torch.equal(a.vals[0], b.vals[0])
