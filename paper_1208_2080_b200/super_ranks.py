"""One process per GPU for the super-lattice decomposition (PAPER.md:54 "one MPI rank per GPU", :62-84).

Rank r owns piece r of the gx x gy super-lattice (`sw_create_super_rank`).  The ranks exchange the CUDA IPC handles of
their pieces once (all_gather over torch.distributed), after which every kernel reaches its neighbours' memory directly
(NVLink P2P between GPUs).  A sweep is three phases with a barrier of the process group after each -- stage 1 inside the
pieces, stage 2 between them, resolve + flatten + flip -- which is all that remains of the paper's per-round exchange of
boundary buffers and termination flags.  Only this control plane lives here; every step of the path runs
in the kernels behind the C ABI (`backend` is the ctypes binding; the CPU tests inject a recording stand-in to check the
lock-step protocol with gloo).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import binding as sw

IPC_HANDLE_BYTES = 64


class LibBackend:
    """The C ABI calls a rank makes (include/sw.h, 'one process per GPU')."""

    def __init__(self, L, q, K, seed, gx, gy, piece):
        self.q, self.N = int(q), int(L) * int(L)
        self._h = C.c_void_p()
        l = sw.lib()
        l.sw_create_super_rank.argtypes = [C.POINTER(C.c_void_p), C.c_uint32, C.c_uint32, C.c_double, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        l.sw_super_ipc_export.argtypes = [C.c_void_p, C.c_void_p]
        l.sw_super_ipc_import.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p]
        l.sw_super_phase.argtypes = [C.c_void_p, C.c_int]
        l.sw_super_measure_phase.argtypes = [C.c_void_p, C.c_int, C.c_uint32, C.POINTER(C.c_uint64)]
        rc = l.sw_create_super_rank(C.byref(self._h), int(L), int(q), float(K), int(seed), int(gx), int(gy), int(piece))
        if rc != sw.OK:
            self._h = C.c_void_p()
            raise sw.SwError(rc, "sw_create_super_rank")

    def _chk(self, rc, what):
        if rc != sw.OK:
            msg = sw.lib().sw_super_last_error(self._h)
            raise sw.SwError(rc, what, msg.decode() if msg else "")

    def export_handle(self) -> bytes:
        buf = (C.c_uint8 * IPC_HANDLE_BYTES)()
        self._chk(sw.lib().sw_super_ipc_export(self._h, buf), "sw_super_ipc_export")
        return bytes(buf)

    def import_handle(self, piece, handle: bytes):
        buf = (C.c_uint8 * IPC_HANDLE_BYTES).from_buffer_copy(handle)
        self._chk(sw.lib().sw_super_ipc_import(self._h, int(piece), buf), "sw_super_ipc_import")

    def init(self, mode):
        self._chk(sw.lib().sw_super_init(self._h, {"ordered": 0, "random": 1}.get(mode, mode)), "sw_super_init")

    def set_state(self, spins, t):
        s = np.ascontiguousarray(spins, dtype=np.uint8).reshape(-1)
        self._chk(sw.lib().sw_super_set_state(self._h, s.ctypes.data, int(t)), "sw_super_set_state")

    def phase(self, k):
        self._chk(sw.lib().sw_super_phase(self._h, int(k)), "sw_super_phase")

    def synchronize(self):
        self._chk(sw.lib().sw_super_synchronize(self._h), "sw_super_synchronize")

    def measure_phase(self, k, what):
        part = (C.c_uint64 * (3 + self.q))()
        self._chk(sw.lib().sw_super_measure_phase(self._h, int(k), int(what), part), "sw_super_measure_phase")
        return [int(v) for v in part]

    def get(self, what):
        """The local piece's part of a whole-lattice array (the rest is zero)."""
        out = np.zeros(self.N, dtype=np.uint32 if what == "labels" else np.uint8)
        fn = {"spins": sw.lib().sw_super_get_spins, "labels": sw.lib().sw_super_get_labels, "bonds": sw.lib().sw_super_get_bonds}[what]
        self._chk(fn(self._h, out.ctypes.data), f"sw_super_get_{what}")
        return out

    def stats(self):
        """sw_super_get_stats of this rank's context (the counters cover the local piece's share of the work)."""
        st = sw.SuperStats()
        self._chk(sw.lib().sw_super_get_stats(self._h, C.byref(st)), "sw_super_get_stats")
        return {f: int(getattr(st, f)) for f, _ in sw.SuperStats._fields_}

    def close_imported(self):
        """Unmap the other ranks' pieces (sw_super_ipc_close_all); the context can only be closed afterwards."""
        if self._h:
            self._chk(sw.lib().sw_super_ipc_close_all(self._h), "sw_super_ipc_close_all")

    def close(self):
        if self._h:
            sw.lib().sw_super_destroy(self._h)
            self._h = C.c_void_p()


class SuperLatticeRanks:
    """Collective object: every rank of the process group constructs it and makes the same calls in the same order."""

    def __init__(self, L, q, K, seed, gx, gy, backend=None):
        import torch
        import torch.distributed as dist
        self._torch, self._dist = torch, dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        if self.world != gx * gy:
            raise ValueError(f"the super-lattice has {gx * gy} pieces but the process group has {self.world} ranks")
        self.L, self.q, self.N = int(L), int(q), int(L) * int(L)
        self.backend = backend if backend is not None else LibBackend(L, q, K, seed, gx, gy, self.rank)
        # exchange the IPC handles: 64 bytes per rank
        mine = torch.frombuffer(bytearray(self.backend.export_handle()), dtype=torch.uint8).clone()
        everyone = [torch.zeros(IPC_HANDLE_BYTES, dtype=torch.uint8) for _ in range(self.world)]
        dist.all_gather(everyone, mine)
        for piece, h in enumerate(everyone):
            if piece != self.rank:
                self.backend.import_handle(piece, bytes(h.numpy().tobytes()))
        dist.barrier()

    def _step(self):
        """End of a phase: my kernels are done, and so are everyone else's."""
        self.backend.synchronize()
        self._dist.barrier()

    def init(self, mode):
        self.backend.init(mode)
        self._step()

    def set_state(self, spins, t):
        """Every rank loads its own piece of `spins`.  If any rank's piece is refused (a spin >= q), EVERY rank raises:
        the ranks agree on the outcome before the barrier, so no rank is left waiting for one that has already given up."""
        torch, dist = self._torch, self._dist
        err = None
        try:
            self.backend.set_state(spins, t)
        except Exception as e:                               # noqa: BLE001 -- reported below, on every rank
            err = e
        failed = torch.tensor([0 if err is None else 1], dtype=torch.int32)
        dist.all_reduce(failed, op=dist.ReduceOp.SUM)
        if int(failed.item()):
            if err is not None:
                raise err
            raise sw.SwError(sw.ERR_INVALID_ARG, "sw_super_set_state", f"refused on {int(failed.item())} other rank(s)")
        self._step()

    def sweep(self, n=1):
        for _ in range(int(n)):
            for phase in (0, 1, 2):
                self.backend.phase(phase)
                self._step()

    def measure(self, what=sw.OBS_ALL):
        torch, dist = self._torch, self._dist
        part = None
        for phase in (0, 1, 2):
            part = self.backend.measure_phase(phase, what)
            self._step()
        # (the counts of a 2^32-site lattice exceed int64's positive range only in theory: energy_bonds <= 2^33)
        sums = torch.tensor(part, dtype=torch.int64)
        big = torch.tensor([part[2]], dtype=torch.int64)
        dist.all_reduce(sums, op=dist.ReduceOp.SUM)
        dist.all_reduce(big, op=dist.ReduceOp.MAX)
        row = [int(v) for v in sums]
        row[2] = int(big.item())
        if row[1] == 1:
            row[2] = self.N
        return {"energy_bonds": row[0], "n_clusters": row[1], "largest_cluster": row[2], "mag_counts": row[3:]}

    def gather(self, what):
        """The whole-lattice array on every rank (each rank contributes its piece)."""
        torch, dist = self._torch, self._dist
        local = self.backend.get(what)
        t = torch.from_numpy(local.astype(np.int64))
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return t.numpy().astype(local.dtype)

    def close(self):
        """Tear-down in three steps: every rank unmaps the pieces it imported, THEN (barrier) every rank frees its own.
        Freeing an exported piece while another process still has it mapped is undefined behaviour in CUDA IPC."""
        self._dist.barrier()                                 # nobody is still inside a phase
        self.backend.close_imported()
        self._dist.barrier()                                 # nobody has my piece mapped any more
        self.backend.close()
