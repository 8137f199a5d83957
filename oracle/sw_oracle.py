"""ctypes wrapper of the CPU oracle (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this.  It never imports the CUDA package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

ISING, POTTS, XY, CLOCK = 0, 1, 2, 3

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.swo_create.restype = C.c_void_p
        L.swo_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_uint64]
        L.swo_destroy.argtypes = [C.c_void_p]
        L.swo_step.argtypes = [C.c_void_p, C.c_int]
        L.swo_observables.argtypes = [C.c_void_p] + [C.POINTER(C.c_double)] * 4
        L.swo_counts.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.c_int]
        L.swo_num_sites.restype = C.c_size_t
        L.swo_num_sites.argtypes = [C.c_void_p]
        L.swo_step_index.restype = C.c_uint64
        L.swo_step_index.argtypes = [C.c_void_p]
        L.swo_get_spins.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        L.swo_set_spins.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_uint64]
        L.swo_get_bonds.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        L.swo_get_labels.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        L.swo_get_xy_dir.argtypes = [C.c_void_p] + [C.POINTER(C.c_float)] * 3
        L.swo_force_xy_phi.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.swo_run_series.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 6
        L.swo_clock_hist.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.swo_get_clock_mirror.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
        L.swo_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        _lib = L
    return _lib


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().swo_philox4x32_10(c, k, o)
    return [int(x) for x in o]


_SPIN_DTYPE = {ISING: np.int8, POTTS: np.uint8, XY: np.float32, CLOCK: np.uint16}


class Oracle:
    def __init__(self, dim, L, model, q, beta, seed):
        self._h = lib().swo_create(dim, L, model, q, float(beta), int(seed))
        if not self._h:
            raise ValueError("swo_create rejected the arguments")
        self.dim, self.L, self.model, self.q, self.beta, self.seed = dim, L, model, q, beta, seed
        self.N = int(lib().swo_num_sites(self._h))

    def close(self):
        if self._h:
            lib().swo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def t(self):
        return int(lib().swo_step_index(self._h))

    def step(self, n=1):
        if lib().swo_step(self._h, int(n)) != 0:
            raise RuntimeError("swo_step failed")

    def observables(self):
        v = [C.c_double() for _ in range(4)]
        lib().swo_observables(self._h, *[C.byref(x) for x in v])
        return tuple(x.value for x in v)

    def counts(self):
        n = self.q if self.model == POTTS else 1
        e = C.c_int64()
        m = (C.c_int64 * n)()
        if lib().swo_counts(self._h, C.byref(e), m, n) != 0:
            raise RuntimeError("swo_counts: not defined for this model")
        return int(e.value), [int(x) for x in m]

    def spins(self):
        a = np.empty(self.N, dtype=_SPIN_DTYPE[self.model])
        assert lib().swo_get_spins(self._h, a.ctypes.data, a.nbytes) == 0
        return a

    def set_spins(self, a, step):
        a = np.ascontiguousarray(a, dtype=_SPIN_DTYPE[self.model])
        assert a.size == self.N
        assert lib().swo_set_spins(self._h, a.ctypes.data, a.nbytes, int(step)) == 0

    def bonds(self):
        a = np.empty(self.N, dtype=np.uint8)
        assert lib().swo_get_bonds(self._h, a.ctypes.data, a.nbytes) == 0
        return a

    def labels(self):
        a = np.empty(self.N, dtype=np.uint32)
        assert lib().swo_get_labels(self._h, a.ctypes.data, a.nbytes) == 0
        return a

    def clock_hist(self):
        D = np.zeros(self.q, dtype=np.int64)
        n = np.zeros(self.q, dtype=np.int64)
        assert lib().swo_clock_hist(self._h, D.ctypes.data, n.ctypes.data, self.q) == 0
        return D, n

    def clock_mirror(self):
        m = C.c_int()
        assert lib().swo_get_clock_mirror(self._h, C.byref(m)) == 0
        return int(m.value)

    def xy_dir(self):
        v = [C.c_float() for _ in range(3)]
        assert lib().swo_get_xy_dir(self._h, *[C.byref(x) for x in v]) == 0
        return tuple(np.float32(x.value) for x in v)

    def force_xy_phi(self, enable, phi=0.0):
        assert lib().swo_force_xy_phi(self._h, int(bool(enable)), float(phi)) == 0

    def run_series(self, n):
        """n steps; returns dict of per-step series (after each step)."""
        out = {k: np.empty(n, dtype=np.float64) for k in ("E", "M", "M2", "n_active", "n_clusters", "sum_nc2")}
        assert lib().swo_run_series(self._h, int(n), *[out[k].ctypes.data for k in
                                                       ("E", "M", "M2", "n_active", "n_clusters", "sum_nc2")]) == 0
        return out
