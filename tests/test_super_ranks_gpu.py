"""One process per piece, for real: two (and four) processes, each owning one piece of the super-lattice in its own CUDA
context, reaching the other pieces through CUDA IPC -- needs a B200, `-m gpu`.  The box has one GPU, so all ranks use
device 0 (the kernels never wait on another rank inside a launch: the phases are separated by host-side barriers, so
sharing the device is safe); across GPUs the same pointers go over NVLink.  Result: bit-identical to the oracle."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, L, q, K, gx, gy, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        from paper_1208_2080_b200.super_ranks import SuperLatticeRanks
        sim = SuperLatticeRanks(L, q, K, 1, gx, gy)
        sim.init("random")
        res = []
        for n in (1, 2):
            sim.sweep(n)
            m = sim.measure()
            arrays = {w: sim.gather(w) for w in ("bonds", "labels", "spins")}
            if rank == 0:
                res.append((m, arrays))
        if rank == 0:
            out["res"] = res
        sim.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("gx,gy", [(2, 1), (2, 2)])
def test_one_process_per_piece_matches_the_oracle(gx, gy):
    from oracle.binding import Oracle
    from paper_1208_2080_b200 import workloads as wl
    L, q = 512, 2
    K = wl.k_critical(q)
    world = gx * gy
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), L, q, K, gx, gy, out), nprocs=world, join=True)
        res = out["res"]
    cpu = Oracle(L, q, K, 1)
    cpu.init("random")
    for (m, arrays), n in zip(res, (1, 2)):
        cpu.sweep(n)
        assert np.array_equal(arrays["bonds"], cpu.get_bonds())
        assert np.array_equal(arrays["labels"], cpu.get_labels())
        assert np.array_equal(arrays["spins"], cpu.get_spins())
        assert m == cpu.measure()
