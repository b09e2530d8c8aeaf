"""ctypes binding of the XY part of oracle/libsw_oracle.so (sw_xy_oracle.h) -- TEST INFRASTRUCTURE, not product."""
import ctypes as C

import numpy as np

from . import binding as _b

_ready = False


def lib():
    global _ready
    l = _b.lib()
    if not _ready:
        vp, dp, u64p = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_uint64)
        l.swo_xy_reflection.argtypes = [C.c_uint64, C.c_uint32, dp]; l.swo_xy_reflection.restype = None
        l.swo_xy_projection.argtypes = [dp, dp]; l.swo_xy_projection.restype = C.c_double
        l.swo_xy_bond_threshold.argtypes = [C.c_double, C.c_double, C.c_double]; l.swo_xy_bond_threshold.restype = C.c_uint64
        l.swo_xy_reflect.argtypes = [dp, dp]; l.swo_xy_reflect.restype = None
        l.swo_xy_init_spin.argtypes = [C.c_uint64, C.c_uint64, dp]; l.swo_xy_init_spin.restype = None
        l.swo_xy_create.argtypes = [C.POINTER(vp), C.c_uint32, C.c_double, C.c_uint64]; l.swo_xy_create.restype = C.c_int
        l.swo_xy_init.argtypes = [vp, C.c_int]; l.swo_xy_init.restype = C.c_int
        l.swo_xy_set_state.argtypes = [vp, vp, C.c_uint64]; l.swo_xy_set_state.restype = C.c_int
        l.swo_xy_sweep.argtypes = [vp, C.c_uint64]; l.swo_xy_sweep.restype = C.c_int
        l.swo_xy_measure.argtypes = [vp, dp, dp, u64p, u64p]; l.swo_xy_measure.restype = C.c_int
        l.swo_xy_get_spins.argtypes = [vp, vp]; l.swo_xy_get_spins.restype = C.c_int
        l.swo_xy_get_labels.argtypes = [vp, vp]; l.swo_xy_get_labels.restype = C.c_int
        l.swo_xy_get_bonds.argtypes = [vp, vp]; l.swo_xy_get_bonds.restype = C.c_int
        l.swo_xy_get_time.argtypes = [vp, u64p]; l.swo_xy_get_time.restype = C.c_int
        l.swo_xy_destroy.argtypes = [vp]; l.swo_xy_destroy.restype = None
        _ready = True
    return l


def _chk(code, what):
    if code != _b.OK:
        raise _b.OracleError(code, what)


def reflection(seed, t):
    r = (C.c_double * 2)()
    lib().swo_xy_reflection(seed, t, r)
    return float(r[0]), float(r[1])


def projection(s, r):
    return float(lib().swo_xy_projection((C.c_double * 2)(*s), (C.c_double * 2)(*r)))


def bond_threshold(K, a_i, a_j):
    return int(lib().swo_xy_bond_threshold(float(K), float(a_i), float(a_j)))


def reflect(s, r):
    v = (C.c_double * 2)(*s)
    lib().swo_xy_reflect(v, (C.c_double * 2)(*r))
    return float(v[0]), float(v[1])


def init_spin(seed, site):
    v = (C.c_double * 2)()
    lib().swo_xy_init_spin(seed, site, v)
    return float(v[0]), float(v[1])


class OracleXY:
    """One embedded-cluster XY simulation on the CPU oracle (same call names as the product binding)."""

    def __init__(self, L, K, seed):
        self.L, self.K, self.seed = int(L), float(K), int(seed)
        self.N = self.L * self.L
        self._h = C.c_void_p()
        _chk(lib().swo_xy_create(C.byref(self._h), self.L, self.K, self.seed), "xy create")

    def close(self):
        if self._h:
            lib().swo_xy_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init(self, mode):
        _chk(lib().swo_xy_init(self._h, {"ordered": 0, "random": 1}.get(mode, mode)), "xy init")

    def set_state(self, spins, t):
        s = np.ascontiguousarray(spins, dtype=np.float64).reshape(-1)
        assert s.size == 2 * self.N
        _chk(lib().swo_xy_set_state(self._h, s.ctypes.data, int(t)), "xy set_state")

    def sweep(self, n=1):
        _chk(lib().swo_xy_sweep(self._h, int(n)), "xy sweep")

    def measure(self):
        e, nc, big = C.c_double(), C.c_uint64(), C.c_uint64()
        m = (C.c_double * 2)()
        _chk(lib().swo_xy_measure(self._h, C.byref(e), m, C.byref(nc), C.byref(big)), "xy measure")
        return {"energy_sum": float(e.value), "mag": [float(m[0]), float(m[1])], "n_clusters": int(nc.value), "largest_cluster": int(big.value)}

    def get_spins(self):
        out = np.empty((self.N, 2), dtype=np.float64)
        _chk(lib().swo_xy_get_spins(self._h, out.ctypes.data), "xy get_spins")
        return out

    def get_labels(self):
        out = np.empty(self.N, dtype=np.uint32)
        _chk(lib().swo_xy_get_labels(self._h, out.ctypes.data), "xy get_labels")
        return out

    def get_bonds(self):
        out = np.empty(self.N, dtype=np.uint8)
        _chk(lib().swo_xy_get_bonds(self._h, out.ctypes.data), "xy get_bonds")
        return out

    def get_time(self):
        t = C.c_uint64()
        _chk(lib().swo_xy_get_time(self._h, C.byref(t)), "xy get_time")
        return int(t.value)
