"""ctypes binding of oracle/libsw_oracle.so -- TEST INFRASTRUCTURE, not product.

Argument marshalling only; every number comes from sw_oracle.cpp.
"""
import ctypes as C
import math
import os

import numpy as np

from . import build as _build

_lib = None

OK, ERR_INVALID_ARG, ERR_OOM, ERR_STATE = 0, 1, 2, 4
INIT_ORDERED, INIT_RANDOM = 0, 1


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"oracle {what} failed with status {code}")
        self.code = code


def lib():
    global _lib
    if _lib is None:
        # SWO_LIB: tests/oracle_mutations.py points the binding at a deliberately broken copy of the oracle
        l = C.CDLL(os.environ.get("SWO_LIB") or _build.build())
        u8p, u32p, u64p = C.POINTER(C.c_uint8), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
        vp = C.c_void_p
        l.swo_philox4x32_10.argtypes = [u32p, u32p, u32p]; l.swo_philox4x32_10.restype = None
        l.swo_threshold.argtypes = [C.c_double, u64p]; l.swo_threshold.restype = C.c_int
        l.swo_draw_bond.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_int]; l.swo_draw_bond.restype = C.c_uint32
        l.swo_draw_flip.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64]; l.swo_draw_flip.restype = C.c_uint32
        l.swo_draw_init.argtypes = [C.c_uint64, C.c_uint64]; l.swo_draw_init.restype = C.c_uint32
        l.swo_state_from_draw.argtypes = [C.c_uint32, C.c_uint32]; l.swo_state_from_draw.restype = C.c_uint32
        l.swo_label_bonds.argtypes = [C.c_uint32, vp, vp, u64p, u64p]; l.swo_label_bonds.restype = C.c_int
        l.swo_create.argtypes = [C.POINTER(vp), C.c_uint32, C.c_uint32, C.c_double, C.c_uint64]; l.swo_create.restype = C.c_int
        l.swo_init.argtypes = [vp, C.c_int]; l.swo_init.restype = C.c_int
        l.swo_set_state.argtypes = [vp, vp, C.c_uint64]; l.swo_set_state.restype = C.c_int
        l.swo_sweep.argtypes = [vp, C.c_uint64]; l.swo_sweep.restype = C.c_int
        l.swo_measure.argtypes = [vp, u64p, u64p, u64p, u64p]; l.swo_measure.restype = C.c_int
        l.swo_sweep_measure.argtypes = [vp, C.c_uint64, vp]; l.swo_sweep_measure.restype = C.c_int
        l.swo_get_spins.argtypes = [vp, vp]; l.swo_get_spins.restype = C.c_int
        l.swo_get_labels.argtypes = [vp, vp]; l.swo_get_labels.restype = C.c_int
        l.swo_get_bonds.argtypes = [vp, vp]; l.swo_get_bonds.restype = C.c_int
        l.swo_get_threshold.argtypes = [vp, u64p]; l.swo_get_threshold.restype = C.c_int
        l.swo_get_time.argtypes = [vp, u64p]; l.swo_get_time.restype = C.c_int
        l.swo_destroy.argtypes = [vp]; l.swo_destroy.restype = None
        _lib = l
    return _lib


def _chk(code, what):
    if code != OK:
        raise OracleError(code, what)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().swo_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def threshold(K):
    T = C.c_uint64()
    _chk(lib().swo_threshold(float(K), C.byref(T)), "threshold")
    return int(T.value)


def draw_bond(seed, t, site, direction):
    return int(lib().swo_draw_bond(seed, t, site, direction))


def draw_flip(seed, t, root):
    return int(lib().swo_draw_flip(seed, t, root))


def draw_init(seed, site):
    return int(lib().swo_draw_init(seed, site))


def state_from_draw(w, q):
    return int(lib().swo_state_from_draw(w, q))


def label_bonds(bonds):
    """bonds: (L, L) or (L*L,) uint8, bit0 = right, bit1 = down.  Returns (labels, n_clusters, largest)."""
    b = np.ascontiguousarray(bonds, dtype=np.uint8).reshape(-1)
    L = math.isqrt(b.size)
    assert L * L == b.size
    labels = np.empty(b.size, dtype=np.uint32)
    nc, big = C.c_uint64(), C.c_uint64()
    _chk(lib().swo_label_bonds(L, b.ctypes.data, labels.ctypes.data, C.byref(nc), C.byref(big)), "label_bonds")
    return labels, int(nc.value), int(big.value)


class Oracle:
    """One Swendsen-Wang simulation on the CPU oracle (same call names as the product binding)."""

    def __init__(self, L, q, K, seed):
        self.L, self.q, self.K, self.seed = int(L), int(q), float(K), int(seed)
        self.N = self.L * self.L
        self._h = C.c_void_p()
        _chk(lib().swo_create(C.byref(self._h), self.L, self.q, self.K, self.seed), "create")

    def close(self):
        if self._h:
            lib().swo_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init(self, mode):
        _chk(lib().swo_init(self._h, {"ordered": 0, "random": 1}.get(mode, mode)), "init")

    def set_state(self, spins, t):
        s = np.ascontiguousarray(spins, dtype=np.uint8).reshape(-1)
        assert s.size == self.N
        _chk(lib().swo_set_state(self._h, s.ctypes.data, int(t)), "set_state")

    def sweep(self, n=1):
        _chk(lib().swo_sweep(self._h, int(n)), "sweep")

    def measure(self):
        e, nc, big = C.c_uint64(), C.c_uint64(), C.c_uint64()
        mag = (C.c_uint64 * self.q)()
        _chk(lib().swo_measure(self._h, C.byref(e), mag, C.byref(nc), C.byref(big)), "measure")
        return {"energy_bonds": int(e.value), "mag_counts": [int(v) for v in mag],
                "n_clusters": int(nc.value), "largest_cluster": int(big.value)}

    def sweep_measure(self, n):
        """n x (sweep, measure); columns: energy_bonds, n_clusters, largest_cluster, mag_counts[q]."""
        out = np.zeros((int(n), 3 + self.q), dtype=np.uint64)
        _chk(lib().swo_sweep_measure(self._h, int(n), out.ctypes.data), "sweep_measure")
        return out

    def get_spins(self):
        out = np.empty(self.N, dtype=np.uint8)
        _chk(lib().swo_get_spins(self._h, out.ctypes.data), "get_spins")
        return out

    def get_labels(self):
        out = np.empty(self.N, dtype=np.uint32)
        _chk(lib().swo_get_labels(self._h, out.ctypes.data), "get_labels")
        return out

    def get_bonds(self):
        out = np.empty(self.N, dtype=np.uint8)
        _chk(lib().swo_get_bonds(self._h, out.ctypes.data), "get_bonds")
        return out

    def get_threshold(self):
        T = C.c_uint64()
        _chk(lib().swo_get_threshold(self._h, C.byref(T)), "get_threshold")
        return int(T.value)

    def get_time(self):
        t = C.c_uint64()
        _chk(lib().swo_get_time(self._h, C.byref(t)), "get_time")
        return int(t.value)
