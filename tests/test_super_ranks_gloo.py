"""The one-process-per-GPU control plane of the super-lattice decomposition on CPU: world_size 2 (and 4), gloo, 127.0.0.1.

No CUDA here: the C ABI calls a rank makes are replaced by a recording stand-in, and what is checked is the protocol --
every rank imports every other rank's IPC handle exactly once, the three phases of every sweep run in lock step (no rank
enters phase k + 1 before all ranks have finished phase k), and the partial rows of a measurement are combined with sums
and, for the largest cluster, a maximum."""
import os
import socket
import time

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1208_2080_b200.super_ranks import IPC_HANDLE_BYTES, SuperLatticeRanks


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class RecordingBackend:
    def __init__(self, rank, q, log):
        self.rank, self.q, self.log, self.imported = rank, q, log, {}

    def _rec(self, what):
        self.log.append((time.monotonic(), self.rank, "begin", what))
        time.sleep(0.002 * (self.rank + 1))                  # ranks finish at different times
        self.log.append((time.monotonic(), self.rank, "end", what))

    def export_handle(self):
        return bytes([self.rank]) * IPC_HANDLE_BYTES

    def import_handle(self, piece, handle):
        assert piece not in self.imported and handle == bytes([piece]) * IPC_HANDLE_BYTES
        self.imported[piece] = handle

    def init(self, mode):
        self._rec(("init", mode))

    def phase(self, k):
        self._rec(("phase", k))

    def synchronize(self):
        pass

    def measure_phase(self, k, what):
        self._rec(("measure", k))
        # energy, n_clusters, largest, mag[q]
        return [10 * (self.rank + 1), 3 + self.rank, 100 + 7 * self.rank] + [self.rank + s for s in range(self.q)]

    def set_state(self, spins, t):
        if self.rank == 1 and int(np.max(spins)) >= self.q:
            raise ValueError("spin value >= q on rank 1")
        self._rec(("set_state", int(t)))

    def close_imported(self):
        self._rec("close_imported")

    def close(self):
        self._rec("close")


def _worker(rank, world, port, gx, gy, log, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        be = RecordingBackend(rank, 3, log)
        sim = SuperLatticeRanks(128 * gx, 3, 1.0, 1, gx, gy, backend=be)
        sim.init("random")
        sim.sweep(3)
        out[rank] = (sim.measure(), sorted(be.imported))
        # a state that only rank 1 refuses: every rank must raise (and none may hang in the barrier that follows)
        L = 128 * gx
        try:
            sim.set_state(np.full(L * L, 3, dtype=np.uint8), 5)
            out[("set_state", rank)] = "accepted"
        except Exception as e:                               # noqa: BLE001
            out[("set_state", rank)] = type(e).__name__
        sim.set_state(np.zeros(L * L, dtype=np.uint8), 5)    # the ranks are still in step afterwards
        sim.close()
    finally:
        dist.destroy_process_group()


def _run(gx, gy):
    world = gx * gy
    with mp.Manager() as mgr:
        log, out = mgr.list(), mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), gx, gy, log, out), nprocs=world, join=True)
        return sorted(log), dict(out)


def check(gx, gy):
    world = gx * gy
    log, out = _run(gx, gy)
    for rank in range(world):
        assert out[("set_state", rank)] == ("ValueError" if rank == 1 else "SwError")
        m, imported = out[rank]
        assert imported == [r for r in range(world) if r != rank]
        assert m["energy_bonds"] == 10 * sum(r + 1 for r in range(world))
        assert m["n_clusters"] == sum(3 + r for r in range(world))
        assert m["largest_cluster"] == 100 + 7 * (world - 1)          # a maximum, not a sum
        assert m["mag_counts"] == [sum(r + s for r in range(world)) for s in range(3)]
    # lock step: the steps appear in the same order on every rank, and step k ends everywhere before step k + 1 begins anywhere
    steps = [w for (_, r, kind, w) in log if r == 0 and kind == "begin"]
    in_step = [("init", "random")] + [("phase", k) for _ in range(3) for k in (0, 1, 2)] + [("measure", k) for k in (0, 1, 2)]
    # (rank 0's own piece was accepted both times; the first time it raised all the same, because rank 1 refused)
    assert steps == in_step + [("set_state", 5), ("set_state", 5), "close_imported", "close"]
    steps = in_step
    # tear-down: every rank has unmapped its imports before any rank frees its piece
    assert max(t for (t, r, kind, w) in log if kind == "end" and w == "close_imported") <= \
        min(t for (t, r, kind, w) in log if kind == "begin" and w == "close")
    for i in range(len(steps) - 1):
        ends = [t for (t, r, kind, w) in log if kind == "end" and w == steps[i]]
        later = [j for j, (t, r, kind, w) in enumerate(log) if kind == "begin" and w == steps[i + 1]]
        # several identical step names exist (3 sweeps): compare occurrence by occurrence
        occ = steps[:i + 1].count(steps[i]) - 1
        ends_i = sorted(ends)[occ * world:(occ + 1) * world]
        occ_n = steps[:i + 2].count(steps[i + 1]) - 1
        begins_n = sorted(log[j][0] for j in later)[occ_n * world:(occ_n + 1) * world]
        assert len(ends_i) == world and len(begins_n) == world
        assert max(ends_i) <= min(begins_n), (steps[i], steps[i + 1])


def test_two_ranks_lock_step():
    check(2, 1)


def test_four_ranks_lock_step():
    check(2, 2)
