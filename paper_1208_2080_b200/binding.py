"""Thin ctypes binding of libsw.so (include/sw.h) -- argument marshalling only.

Every step of the sweep runs in the CUDA kernels behind the C ABI.  PyTorch is used for two
things only: the device workspace is a torch uint8 tensor (so the caching allocator owns the
memory) and the kernels are enqueued on torch's current CUDA stream.  There is no CPU fallback:
if libsw.so has not been built or no CUDA device is present, creating a `SwendsenWang` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

OK, ERR_INVALID_ARG, ERR_OOM, ERR_CUDA, ERR_STATE = 0, 1, 2, 3, 4
INIT_ORDERED, INIT_RANDOM = 0, 1
FLAG_DEFAULT, FLAG_FORCE_GENERIC, FLAG_LAZY_LABELS, FLAG_LABEL_EQUIVALENCE = 0, 1, 2, 4
FLAG_WS_CLUSTER_SIZES, FLAG_PASS_COUNTERS, FLAG_NO_CLUSTER_PATH = 8, 16, 32
OBS_ENERGY, OBS_MAG, OBS_CLUSTERS, OBS_LARGEST, OBS_ALL = 1, 2, 4, 8, 15
MAX_KERNEL_SLOTS = 8
_STATUS = {1: "SW_ERR_INVALID_ARG", 2: "SW_ERR_OOM", 3: "SW_ERR_CUDA", 4: "SW_ERR_STATE"}

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libsw.so")
_lib = None

# every symbol include/sw.h declares (tests check that the library exports them all)
SYMBOLS = [
    "sw_create", "sw_create_ex", "sw_workspace_bytes", "sw_create_ws", "sw_destroy", "sw_init",
    "sw_set_state", "sw_set_state_packed", "sw_get_spins_packed", "sw_sweep", "sw_measure", "sw_measure_clusters", "sw_sweep_measure", "sw_sweep_measure_ex", "sw_get_spins", "sw_get_labels",
    "sw_get_bonds", "sw_get_rows", "sw_get_threshold", "sw_get_time", "sw_synchronize",
    "sw_get_stats", "sw_profile_begin", "sw_profile_end", "sw_profile_series", "sw_kernel_name", "sw_last_error",
    "sw_version",
    "sw_create_super", "sw_super_destroy", "sw_super_init", "sw_super_set_state", "sw_super_sweep", "sw_super_measure",
    "sw_super_get_spins", "sw_super_get_labels", "sw_super_get_bonds", "sw_super_get_time", "sw_super_synchronize",
    "sw_super_get_stats", "sw_super_last_error",
    "sw_create_super_rank", "sw_super_ipc_export", "sw_super_ipc_import", "sw_super_ipc_close_all", "sw_super_phase", "sw_super_measure_phase",
    "sw_xy_create", "sw_xy_destroy", "sw_xy_init", "sw_xy_set_state", "sw_xy_sweep", "sw_xy_measure", "sw_xy_get_spins",
    "sw_xy_get_labels", "sw_xy_get_bonds", "sw_xy_get_reflection", "sw_xy_get_time", "sw_xy_last_error",
    "sw_cluster_stats_static", "sw_static_max_sites", "sw_static_last_error",
]


class SwError(RuntimeError):
    def __init__(self, code, what, detail=""):
        super().__init__(f"{what}: {_STATUS.get(code, code)}" + (f" ({detail})" if detail else ""))
        self.code = code


class Stats(C.Structure):
    _fields_ = [("path", C.c_uint32), ("tile_w", C.c_uint32), ("tile_h", C.c_uint32),
                ("kernels_per_sweep", C.c_uint32), ("kernel_launches", C.c_uint64),
                ("device_bytes", C.c_uint64), ("sweeps", C.c_uint64),
                ("le_rounds_last", C.c_uint64), ("le_rounds_total", C.c_uint64),
                ("merge_links", C.c_uint64), ("merge_retries", C.c_uint64), ("merge_hops", C.c_uint64),
                ("chase_hops", C.c_uint64), ("max_merge_depth", C.c_uint32), ("max_chase_depth", C.c_uint32),
                ("bytes_moved", C.c_uint64)]


class SuperStats(C.Structure):
    _fields_ = [("gx", C.c_uint32), ("gy", C.c_uint32), ("piece_w", C.c_uint32), ("piece_h", C.c_uint32), ("devices", C.c_uint32),
                ("sweeps", C.c_uint64), ("kernel_launches", C.c_uint64), ("device_bytes", C.c_uint64),
                ("boundary_sites_per_piece", C.c_uint64), ("inter_links", C.c_uint64), ("inter_hops", C.c_uint64),
                ("inter_retries", C.c_uint64), ("resolved_links", C.c_uint64)]


def lib():
    """Load libsw.so (built by `python -m paper_1208_2080_b200.build`); raise if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise SwError(ERR_CUDA, "libsw.so not found",
                      f"{LIB_PATH}; build it with `python -m paper_1208_2080_b200.build`")
    l = C.CDLL(LIB_PATH)
    vp, u64p = C.c_void_p, C.POINTER(C.c_uint64)
    l.sw_create.argtypes = [C.POINTER(vp), C.c_uint32, C.c_uint32, C.c_double, C.c_uint64]
    l.sw_create_ex.argtypes = [C.POINTER(vp), C.c_uint32, C.c_uint32, C.c_double, C.c_uint64, C.c_uint32]
    l.sw_workspace_bytes.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32]
    l.sw_workspace_bytes.restype = C.c_size_t
    l.sw_create_ws.argtypes = [C.POINTER(vp), C.c_uint32, C.c_uint32, C.c_double, C.c_uint64, C.c_uint32,
                               vp, C.c_size_t, vp]
    l.sw_destroy.argtypes = [vp]; l.sw_destroy.restype = None
    l.sw_init.argtypes = [vp, C.c_int]
    l.sw_set_state.argtypes = [vp, vp, C.c_uint64]
    l.sw_set_state_packed.argtypes = [vp, vp, C.c_uint32, C.c_uint64]
    l.sw_get_spins_packed.argtypes = [vp, vp, C.c_uint32]
    l.sw_sweep.argtypes = [vp, C.c_uint64]
    l.sw_measure.argtypes = [vp, u64p, u64p, u64p, u64p]
    l.sw_measure_clusters.argtypes = [vp, u64p, u64p, u64p]
    l.sw_sweep_measure.argtypes = [vp, C.c_uint64, vp]
    l.sw_sweep_measure_ex.argtypes = [vp, C.c_uint64, vp, C.c_uint32]
    l.sw_get_spins.argtypes = [vp, vp]
    l.sw_get_labels.argtypes = [vp, vp]
    l.sw_get_bonds.argtypes = [vp, vp]
    l.sw_get_rows.argtypes = [vp, C.c_int, C.c_uint32, C.c_uint32, vp]
    l.sw_get_threshold.argtypes = [vp, u64p]
    l.sw_get_time.argtypes = [vp, u64p]
    l.sw_synchronize.argtypes = [vp]
    l.sw_get_stats.argtypes = [vp, C.POINTER(Stats)]
    l.sw_profile_begin.argtypes = [vp]
    l.sw_profile_end.argtypes = [vp, C.POINTER(C.c_double), u64p]
    l.sw_profile_series.argtypes = [vp, C.POINTER(C.c_double), C.c_uint64, u64p]
    l.sw_kernel_name.argtypes = [vp, C.c_int]; l.sw_kernel_name.restype = C.c_char_p
    l.sw_last_error.argtypes = [vp]; l.sw_last_error.restype = C.c_char_p
    l.sw_version.argtypes = []; l.sw_version.restype = C.c_char_p
    l.sw_create_super.argtypes = [C.POINTER(vp), C.c_uint32, C.c_uint32, C.c_double, C.c_uint64, C.c_uint32, C.c_uint32, C.POINTER(C.c_int)]
    l.sw_super_destroy.argtypes = [vp]; l.sw_super_destroy.restype = None
    l.sw_super_init.argtypes = [vp, C.c_int]
    l.sw_super_set_state.argtypes = [vp, vp, C.c_uint64]
    l.sw_super_sweep.argtypes = [vp, C.c_uint64]
    l.sw_super_measure.argtypes = [vp, u64p, u64p, u64p, u64p]
    l.sw_super_get_spins.argtypes = [vp, vp]
    l.sw_super_get_labels.argtypes = [vp, vp]
    l.sw_super_get_bonds.argtypes = [vp, vp]
    l.sw_super_get_time.argtypes = [vp, u64p]
    l.sw_super_synchronize.argtypes = [vp]
    l.sw_super_get_stats.argtypes = [vp, C.POINTER(SuperStats)]
    l.sw_super_last_error.argtypes = [vp]; l.sw_super_last_error.restype = C.c_char_p
    l.sw_super_ipc_close_all.argtypes = [vp]
    dp = C.POINTER(C.c_double)
    l.sw_xy_create.argtypes = [C.POINTER(vp), C.c_uint32, C.c_double, C.c_uint64]
    l.sw_xy_destroy.argtypes = [vp]; l.sw_xy_destroy.restype = None
    l.sw_xy_init.argtypes = [vp, C.c_int]
    l.sw_xy_set_state.argtypes = [vp, vp, C.c_uint64]
    l.sw_xy_sweep.argtypes = [vp, C.c_uint64]
    l.sw_xy_measure.argtypes = [vp, dp, dp, u64p, u64p]
    l.sw_xy_get_spins.argtypes = [vp, vp]
    l.sw_xy_get_labels.argtypes = [vp, vp]
    l.sw_xy_get_bonds.argtypes = [vp, vp]
    l.sw_xy_get_reflection.argtypes = [vp, dp]
    l.sw_xy_get_time.argtypes = [vp, u64p]
    l.sw_xy_last_error.argtypes = [vp]; l.sw_xy_last_error.restype = C.c_char_p
    l.sw_cluster_stats_static.argtypes = [vp, C.c_uint64, vp, vp]
    l.sw_static_max_sites.argtypes = []; l.sw_static_max_sites.restype = C.c_uint64
    l.sw_static_last_error.argtypes = []; l.sw_static_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        getattr(l, name)                         # AttributeError here = the library is stale
    _lib = l
    return l


def workspace_bytes(L, q, flags=FLAG_DEFAULT):
    return int(lib().sw_workspace_bytes(L, q, flags))


def static_max_sites():
    return int(lib().sw_static_max_sites())


def cluster_stats_static(dev_labels_ptr, n_sites, dev_out_ptr, cuda_stream=0):
    """sw_cluster_stats_static: cluster count, largest cluster and sum of squared sizes of `n_sites` canonical labels,
    for callers that must not allocate on the device (the counters are a fixed array inside libsw.so; at most
    static_max_sites() sites).  All three pointers are raw DEVICE addresses / a cudaStream_t as integers; the result
    (uint64[4] at dev_out_ptr) is ready once the stream has been synchronised.  Calls on one GPU share the counters:
    keep them on one stream."""
    rc = lib().sw_cluster_stats_static(C.c_void_p(dev_labels_ptr), int(n_sites), C.c_void_p(dev_out_ptr), C.c_void_p(cuda_stream))
    if rc != OK:
        msg = lib().sw_static_last_error()
        raise SwError(rc, "sw_cluster_stats_static", msg.decode() if msg else "")


class SwendsenWang:
    """One lattice on one GPU.  Method names follow include/sw.h without the `sw_` prefix."""

    def __init__(self, L, q, K, seed, *, flags=FLAG_DEFAULT, device=None, use_torch=True):
        self.L, self.q, self.K, self.seed, self.flags = int(L), int(q), float(K), int(seed), int(flags)
        self.N = self.L * self.L
        self._h = C.c_void_p()
        self._ws = None
        l = lib()
        if use_torch:
            import torch
            if not torch.cuda.is_available():
                raise SwError(ERR_CUDA, "sw_create_ws", "no CUDA device: the library has no CPU path")
            dev = torch.device("cuda", torch.cuda.current_device() if device is None else device)
            nbytes = workspace_bytes(self.L, self.q, self.flags)
            if nbytes == 0:
                raise SwError(ERR_INVALID_ARG, "sw_workspace_bytes")
            with torch.cuda.device(dev):
                self._ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
                self._stream = torch.cuda.current_stream(dev)
                rc = l.sw_create_ws(C.byref(self._h), self.L, self.q, self.K, self.seed, self.flags,
                                    C.c_void_p(self._ws.data_ptr()), nbytes, C.c_void_p(self._stream.cuda_stream))
        else:
            rc = l.sw_create_ex(C.byref(self._h), self.L, self.q, self.K, self.seed, self.flags)
        if rc != OK:
            self._h = C.c_void_p()
            raise SwError(rc, "sw_create")

    # -- life cycle
    def close(self):
        if self._h:
            lib().sw_destroy(self._h)
            self._h = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, what):
        if rc != OK:
            msg = lib().sw_last_error(self._h)
            raise SwError(rc, what, msg.decode() if msg else "")

    # -- state
    def init(self, mode):
        self._chk(lib().sw_init(self._h, {"ordered": INIT_ORDERED, "random": INIT_RANDOM}.get(mode, mode)), "sw_init")

    def set_state(self, spins, t):
        s = np.ascontiguousarray(spins, dtype=np.uint8).reshape(-1)
        if s.size != self.N:
            raise SwError(ERR_INVALID_ARG, "sw_set_state", "wrong number of spins")
        self._chk(lib().sw_set_state(self._h, s.ctypes.data, int(t)), "sw_set_state")

    def set_state_ptr(self, host_ptr, t):
        """As set_state, from a raw host pointer (e.g. a pinned torch tensor's data_ptr())."""
        self._chk(lib().sw_set_state(self._h, C.c_void_p(host_ptr), int(t)), "sw_set_state")

    def set_state_packed(self, packed, bits, t):
        """packed: uint8 array of L*L*bits/8 bytes, or a raw host pointer (int)."""
        if isinstance(packed, int):
            ptr = C.c_void_p(packed)
        else:
            a = np.ascontiguousarray(packed, dtype=np.uint8).reshape(-1)
            if a.size != self.N * int(bits) // 8:
                raise SwError(ERR_INVALID_ARG, "sw_set_state_packed", "wrong number of bytes")
            ptr = C.c_void_p(a.ctypes.data)
        self._chk(lib().sw_set_state_packed(self._h, ptr, int(bits), int(t)), "sw_set_state_packed")

    def get_spins_packed(self, bits, out=None):
        """Returns a uint8 array of L*L*bits/8 bytes; `out` may be a raw host pointer (int) instead."""
        if isinstance(out, int):
            self._chk(lib().sw_get_spins_packed(self._h, C.c_void_p(out), int(bits)), "sw_get_spins_packed")
            return None
        out = np.empty(self.N * int(bits) // 8, dtype=np.uint8) if out is None else out
        self._chk(lib().sw_get_spins_packed(self._h, out.ctypes.data, int(bits)), "sw_get_spins_packed")
        return out

    # -- hot path
    def sweep(self, n=1):
        self._chk(lib().sw_sweep(self._h, int(n)), "sw_sweep")

    def measure(self, energy=True, mag=True, clusters=True, largest=True):
        e, nc, big = C.c_uint64(), C.c_uint64(), C.c_uint64()
        m = (C.c_uint64 * self.q)()
        self._chk(lib().sw_measure(self._h, C.byref(e) if energy else None, m if mag else None,
                                   C.byref(nc) if clusters else None, C.byref(big) if largest else None), "sw_measure")
        out = {}
        if energy: out["energy_bonds"] = int(e.value)
        if mag: out["mag_counts"] = [int(v) for v in m]
        if clusters: out["n_clusters"] = int(nc.value)
        if largest: out["largest_cluster"] = int(big.value)
        return out

    def measure_clusters(self):
        """n_clusters, largest_cluster and sum over clusters of |c|^2 (a Python int: up to 2^64) of the last sweep."""
        nc, big = C.c_uint64(), C.c_uint64()
        sq = (C.c_uint64 * 2)()
        self._chk(lib().sw_measure_clusters(self._h, C.byref(nc), C.byref(big), sq), "sw_measure_clusters")
        return {"n_clusters": int(nc.value), "largest_cluster": int(big.value), "sum_sq": int(sq[0]) + (int(sq[1]) << 64)}

    def sweep_measure(self, n, what=OBS_ALL):
        """n x (sweep, measure); columns: energy_bonds, n_clusters, largest_cluster, mag_counts[q]."""
        out = np.zeros((int(n), 3 + self.q), dtype=np.uint64)
        self._chk(lib().sw_sweep_measure_ex(self._h, int(n), out.ctypes.data, int(what)), "sw_sweep_measure")
        return out

    # -- read-back
    def get_spins(self, out=None):
        out = np.empty(self.N, dtype=np.uint8) if out is None else out
        self._chk(lib().sw_get_spins(self._h, out.ctypes.data), "sw_get_spins")
        return out

    def get_spins_ptr(self, host_ptr):
        self._chk(lib().sw_get_spins(self._h, C.c_void_p(host_ptr)), "sw_get_spins")

    def get_labels(self):
        out = np.empty(self.N, dtype=np.uint32)
        self._chk(lib().sw_get_labels(self._h, out.ctypes.data), "sw_get_labels")
        return out

    def get_bonds(self):
        out = np.empty(self.N, dtype=np.uint8)
        self._chk(lib().sw_get_bonds(self._h, out.ctypes.data), "sw_get_bonds")
        return out

    def get_rows(self, what, y0, nrows):
        code = {"spins": 0, "labels": 1, "bonds": 2}[what]
        out = np.empty(int(nrows) * self.L, dtype=np.uint32 if code == 1 else np.uint8)
        self._chk(lib().sw_get_rows(self._h, code, int(y0), int(nrows), out.ctypes.data), "sw_get_rows")
        return out.reshape(int(nrows), self.L)

    def get_threshold(self):
        T = C.c_uint64()
        self._chk(lib().sw_get_threshold(self._h, C.byref(T)), "sw_get_threshold")
        return int(T.value)

    def get_time(self):
        t = C.c_uint64()
        self._chk(lib().sw_get_time(self._h, C.byref(t)), "sw_get_time")
        return int(t.value)

    def synchronize(self):
        self._chk(lib().sw_synchronize(self._h), "sw_synchronize")

    # -- introspection
    def stats(self):
        s = Stats()
        self._chk(lib().sw_get_stats(self._h, C.byref(s)), "sw_get_stats")
        out = {f: int(getattr(s, f)) for f, _ in Stats._fields_}
        out["path_name"] = {0: "generic", 1: "tiled", 2: "cluster (one persistent launch)"}.get(out["path"], "?")
        return out

    def profile_series(self):
        """Per-sweep device milliseconds of the region closed by the last profile_end()."""
        n = C.c_uint64()
        self._chk(lib().sw_profile_series(self._h, None, 0, C.byref(n)), "sw_profile_series")
        buf = (C.c_double * max(1, n.value))()
        self._chk(lib().sw_profile_series(self._h, buf, n.value, C.byref(n)), "sw_profile_series")
        return [float(buf[i]) for i in range(n.value)]

    def profile_begin(self):
        self._chk(lib().sw_profile_begin(self._h), "sw_profile_begin")

    def profile_end(self):
        ms = (C.c_double * MAX_KERNEL_SLOTS)()
        n = (C.c_uint64 * MAX_KERNEL_SLOTS)()
        self._chk(lib().sw_profile_end(self._h, ms, n), "sw_profile_end")
        self.last_series = self.profile_series()
        out = {}
        for slot in range(MAX_KERNEL_SLOTS):
            name = lib().sw_kernel_name(self._h, slot)
            if name and n[slot]:
                out[name.decode()] = {"ms": float(ms[slot]), "launches": int(n[slot])}
        return out


class SuperLattice:
    """The gx x gy super-lattice decomposition driven from one process; same results as SwendsenWang.

    `devices`: one CUDA device index per piece (row-major, piece (px, py) = devices[py * gx + px]); None = the current
    device for every piece.  Method names follow include/sw.h without the `sw_super_` prefix."""

    def __init__(self, L, q, K, seed, gx, gy, devices=None):
        self.L, self.q, self.K, self.seed, self.gx, self.gy = int(L), int(q), float(K), int(seed), int(gx), int(gy)
        self.N = self.L * self.L
        self._h = C.c_void_p()
        dev = None
        if devices is not None:
            if len(devices) != self.gx * self.gy:
                raise SwError(ERR_INVALID_ARG, "sw_create_super", "one device per piece")
            dev = (C.c_int * len(devices))(*[int(d) for d in devices])
        rc = lib().sw_create_super(C.byref(self._h), self.L, self.q, self.K, self.seed, self.gx, self.gy, dev)
        if rc != OK:
            self._h = C.c_void_p()
            why = lib().sw_super_last_error(None)             # (no context to ask: the reason of this thread's last failed creation)
            raise SwError(rc, "sw_create_super", why.decode() if why else "")

    def close(self):
        if self._h:
            lib().sw_super_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, what):
        if rc != OK:
            msg = lib().sw_super_last_error(self._h)
            raise SwError(rc, what, msg.decode() if msg else "")

    def init(self, mode):
        self._chk(lib().sw_super_init(self._h, {"ordered": INIT_ORDERED, "random": INIT_RANDOM}.get(mode, mode)), "sw_super_init")

    def set_state(self, spins, t):
        s = np.ascontiguousarray(spins, dtype=np.uint8).reshape(-1)
        if s.size != self.N:
            raise SwError(ERR_INVALID_ARG, "sw_super_set_state", "wrong number of spins")
        self._chk(lib().sw_super_set_state(self._h, s.ctypes.data, int(t)), "sw_super_set_state")

    def sweep(self, n=1):
        self._chk(lib().sw_super_sweep(self._h, int(n)), "sw_super_sweep")

    def measure(self, energy=True, mag=True, clusters=True, largest=True):
        e, nc, big = C.c_uint64(), C.c_uint64(), C.c_uint64()
        m = (C.c_uint64 * self.q)()
        self._chk(lib().sw_super_measure(self._h, C.byref(e) if energy else None, m if mag else None,
                                         C.byref(nc) if clusters else None, C.byref(big) if largest else None), "sw_super_measure")
        out = {}
        if energy: out["energy_bonds"] = int(e.value)
        if mag: out["mag_counts"] = [int(v) for v in m]
        if clusters: out["n_clusters"] = int(nc.value)
        if largest: out["largest_cluster"] = int(big.value)
        return out

    def get_spins(self):
        out = np.empty(self.N, dtype=np.uint8)
        self._chk(lib().sw_super_get_spins(self._h, out.ctypes.data), "sw_super_get_spins")
        return out

    def get_labels(self):
        out = np.empty(self.N, dtype=np.uint32)
        self._chk(lib().sw_super_get_labels(self._h, out.ctypes.data), "sw_super_get_labels")
        return out

    def get_bonds(self):
        out = np.empty(self.N, dtype=np.uint8)
        self._chk(lib().sw_super_get_bonds(self._h, out.ctypes.data), "sw_super_get_bonds")
        return out

    def get_time(self):
        t = C.c_uint64()
        self._chk(lib().sw_super_get_time(self._h, C.byref(t)), "sw_super_get_time")
        return int(t.value)

    def synchronize(self):
        self._chk(lib().sw_super_synchronize(self._h), "sw_super_synchronize")

    def stats(self):
        s = SuperStats()
        self._chk(lib().sw_super_get_stats(self._h, C.byref(s)), "sw_super_get_stats")
        return {f: int(getattr(s, f)) for f, _ in SuperStats._fields_}


class XYModel:
    """Embedded-cluster sweeps of the 2D classical XY model; method names follow include/sw.h (`sw_xy_`)."""

    def __init__(self, L, K, seed):
        self.L, self.K, self.seed = int(L), float(K), int(seed)
        self.N = self.L * self.L
        self._h = C.c_void_p()
        rc = lib().sw_xy_create(C.byref(self._h), self.L, self.K, self.seed)
        if rc != OK:
            self._h = C.c_void_p()
            raise SwError(rc, "sw_xy_create")

    def close(self):
        if self._h:
            lib().sw_xy_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, what):
        if rc != OK:
            msg = lib().sw_xy_last_error(self._h)
            raise SwError(rc, what, msg.decode() if msg else "")

    def init(self, mode):
        self._chk(lib().sw_xy_init(self._h, {"ordered": INIT_ORDERED, "random": INIT_RANDOM}.get(mode, mode)), "sw_xy_init")

    def set_state(self, spins, t):
        s = np.ascontiguousarray(spins, dtype=np.float64).reshape(-1)
        if s.size != 2 * self.N:
            raise SwError(ERR_INVALID_ARG, "sw_xy_set_state", "wrong number of spin components")
        self._chk(lib().sw_xy_set_state(self._h, s.ctypes.data, int(t)), "sw_xy_set_state")

    def sweep(self, n=1):
        self._chk(lib().sw_xy_sweep(self._h, int(n)), "sw_xy_sweep")

    def measure(self):
        e, nc, big = C.c_double(), C.c_uint64(), C.c_uint64()
        m = (C.c_double * 2)()
        self._chk(lib().sw_xy_measure(self._h, C.byref(e), m, C.byref(nc), C.byref(big)), "sw_xy_measure")
        return {"energy_sum": float(e.value), "mag": [float(m[0]), float(m[1])], "n_clusters": int(nc.value), "largest_cluster": int(big.value)}

    def get_spins(self):
        out = np.empty((self.N, 2), dtype=np.float64)
        self._chk(lib().sw_xy_get_spins(self._h, out.ctypes.data), "sw_xy_get_spins")
        return out

    def get_labels(self):
        out = np.empty(self.N, dtype=np.uint32)
        self._chk(lib().sw_xy_get_labels(self._h, out.ctypes.data), "sw_xy_get_labels")
        return out

    def get_bonds(self):
        out = np.empty(self.N, dtype=np.uint8)
        self._chk(lib().sw_xy_get_bonds(self._h, out.ctypes.data), "sw_xy_get_bonds")
        return out

    def get_reflection(self):
        r = (C.c_double * 2)()
        self._chk(lib().sw_xy_get_reflection(self._h, r), "sw_xy_get_reflection")
        return float(r[0]), float(r[1])

    def get_time(self):
        t = C.c_uint64()
        self._chk(lib().sw_xy_get_time(self._h, C.byref(t)), "sw_xy_get_time")
        return int(t.value)
