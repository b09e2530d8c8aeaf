"""The N > 1 bookkeeping of bench.py on CPU: world_size 2, gloo backend, 127.0.0.1 rendezvous."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1208_2080_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        units, secs, rate = replicas.aggregate_throughput(100.0 * (rank + 1), 2.0 + rank)   # rank 1 is the slower one
        out[rank] = (units, secs, rate, replicas.replica_seed(1, rank))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_aggregate_over_two_ranks():
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        units, secs, rate, seed = res[rank]
        assert units == 300.0 and secs == 3.0 and abs(rate - 100.0) < 1e-12     # sum of units / max of times
        assert seed == 1 + rank


def test_single_process_passthrough():
    assert replicas.aggregate_throughput(10.0, 2.0) == (10.0, 2.0, 5.0)
