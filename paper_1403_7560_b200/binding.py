"""Thin ctypes binding of libsw_b200 (include/sw.h): argument marshalling only.

Every step of the Swendsen-Wang path (arXiv 1403.7560) runs in the CUDA kernels
behind the C ABI.  PyTorch is used for device memory (the workspace is a torch tensor from the
caching allocator) and for the stream; there is no CPU fallback: if the library cannot be built or
loaded, or no CUDA device is visible, this module raises.
"""
import ctypes as C

import numpy as np

from . import build as _build

ISING, POTTS, XY, CLOCK = 0, 1, 2, 3
SW_OK, SW_EINVAL, SW_ENOMEM, SW_ECUDA, SW_ESTATE = 0, -1, -2, -3, -4

_SPIN_DTYPE = {ISING: np.int8, POTTS: np.uint8, XY: np.float32, CLOCK: np.uint16}

_lib = None


class SwError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libsw_b200 error {code}: {msg}")
        self.code = code


def lib():
    """Load (building if needed) libsw_b200.so and declare the C ABI."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, i32, u64, dbl, sz = C.c_void_p, C.c_int, C.c_uint64, C.c_double, C.c_size_t
    L.sw_create.argtypes = [C.POINTER(vp), i32, i32, i32, i32, dbl, u64]
    L.sw_create_in.argtypes = [C.POINTER(vp), i32, i32, i32, i32, dbl, u64, vp, sz, vp]
    L.sw_workspace_bytes.argtypes = [i32, i32, i32, i32]
    L.sw_workspace_bytes.restype = sz
    L.sw_step.argtypes = [vp, i32]
    L.sw_observables.argtypes = [vp] + [C.POINTER(dbl)] * 4
    L.sw_run_series.argtypes = [vp, i32, vp, vp, vp, vp]
    L.sw_destroy.argtypes = [vp]
    L.sw_last_error.restype = C.c_char_p
    L.sw_num_sites.argtypes = [vp]
    L.sw_num_sites.restype = sz
    L.sw_step_index.argtypes = [vp]
    L.sw_step_index.restype = u64
    L.sw_get_spins.argtypes = [vp, vp, sz]
    L.sw_set_spins.argtypes = [vp, vp, sz, u64]
    L.sw_set_record_bonds.argtypes = [vp, i32]
    L.sw_get_bonds.argtypes = [vp, vp, sz]
    L.sw_get_labels.argtypes = [vp, vp, sz]
    L.sw_get_cluster_stats.argtypes = [vp, C.POINTER(u64), C.POINTER(u64)]
    L.sw_get_counts.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), i32]
    L.sw_get_clock_hist.argtypes = [vp, vp, vp, i32]
    L.sw_get_clock_mirror.argtypes = [vp, C.POINTER(i32)]
    L.sw_get_xy_dir.argtypes = [vp] + [C.POINTER(C.c_float)] * 3
    L.sw_force_xy_phi.argtypes = [vp, i32, dbl]
    L.sw_set_counting.argtypes = [vp, i32]
    L.sw_get_label_stats.argtypes = [vp, C.POINTER(u64), i32]
    L.sw_set_kernel_timing.argtypes = [vp, i32]
    L.sw_get_kernel_times.argtypes = [vp, C.POINTER(dbl), i32, C.POINTER(u64)]
    L.sw_philox_selftest.argtypes = [vp, vp, vp, i32]
    L.sw_info.argtypes = [vp, i32]
    L.sw_info.restype = C.c_longlong
    L.sw_micro_bench.argtypes = [i32, sz, sz, i32, C.POINTER(dbl)]
    L.sw_cluster_stats_static.argtypes = [vp, sz, vp, vp]
    _lib = L
    return _lib


def _check(rc):
    if rc != SW_OK:
        raise SwError(rc, lib().sw_last_error().decode())


def philox_selftest(ctr, key):
    """Philox4x32-10 evaluated by the device code for (count x 4) counters and (count x 2) keys."""
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.empty_like(ctr)
    _check(lib().sw_philox_selftest(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, len(ctr)))
    return out


MICRO_PHILOX_SITE, MICRO_PHILOX_GROUP, MICRO_GATHER = 0, 1, 2
INFO = {"tile_x": 0, "tile_y": 1, "tile_z": 2, "rows_per_thread": 3, "flip_sites_per_thread": 4, "one_cta": 5,
        "launches_per_step": 6, "observables_copy_bytes": 7}


def micro_bench(kind, n, table_words=0, reps=10):
    """sw_micro_bench (include/sw.h): mean milliseconds per launch of one of the micro-benchmark kernels."""
    ms = dbl_()
    _check(lib().sw_micro_bench(int(kind), int(n), int(table_words), int(reps), C.byref(ms)))
    return float(ms.value)


def dbl_():
    return C.c_double()


STATIC_MAX_SITES = 1 << 20   # SW_STATIC_MAX_SITES (include/sw.h)


def cluster_stats_static(device_labels, n, device_out, cuda_stream=0):
    """sw_cluster_stats_static (include/sw.h): number of clusters and sum of squared cluster sizes of n
    canonical labels, with the scratch counters in the library's static device array -- the call
    allocates nothing.  device_labels / device_out are DEVICE addresses (ints, e.g. tensor.data_ptr()) of
    n uint32 / two uint64; cuda_stream a cudaStream_t as int (0 = the legacy default stream).
    Asynchronous; calls share the scratch array, so calls that overlap on the GPU race."""
    _check(lib().sw_cluster_stats_static(C.c_void_p(int(device_labels)), int(n), C.c_void_p(int(device_out)),
                                         C.c_void_p(int(cuda_stream))))


class SwendsenWang:
    """One simulation context: sw_create / sw_step / sw_observables / sw_destroy (include/sw.h).

    use_torch=True (default) places the context in a torch CUDA tensor and on torch's current stream
    (sw_create_in); use_torch=False lets the library cudaMalloc and own a stream (sw_create)."""

    def __init__(self, dim, L, model, q=0, beta=0.0, seed=1, use_torch=True, record_bonds=False):
        self._h = C.c_void_p()
        self._ws = None
        self.dim, self.L, self.model, self.q, self.beta, self.seed = dim, L, model, q, beta, seed
        if use_torch:
            import torch
            if not torch.cuda.is_available():
                raise SwError(SW_ECUDA, "no CUDA device visible (libsw_b200 has no CPU fallback)")
            nbytes = lib().sw_workspace_bytes(dim, L, model, q)
            if nbytes == 0:
                raise SwError(SW_EINVAL, "invalid arguments")
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            ptr = (self._ws.data_ptr() + 255) // 256 * 256
            stream = torch.cuda.current_stream().cuda_stream
            _check(lib().sw_create_in(C.byref(self._h), dim, L, model, q, float(beta), int(seed),
                                      C.c_void_p(ptr), nbytes, C.c_void_p(stream)))
        else:
            _check(lib().sw_create(C.byref(self._h), dim, L, model, q, float(beta), int(seed)))
        self.N = int(lib().sw_num_sites(self._h))
        if record_bonds:
            self.record_bonds(True)

    def info(self):
        """Launch geometry of this context (sw_info)."""
        return {k: int(lib().sw_info(self._h, v)) for k, v in INFO.items()}

    def record_bonds(self, enable):
        """Steps after this call also store the bond bytes (needed by bonds())."""
        _check(lib().sw_set_record_bonds(self._h, int(bool(enable))))

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

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def t(self):
        return int(lib().sw_step_index(self._h))

    def step(self, n=1):
        _check(lib().sw_step(self._h, int(n)))

    def observables(self):
        v = [C.c_double() for _ in range(4)]
        _check(lib().sw_observables(self._h, *[C.byref(x) for x in v]))
        return tuple(x.value for x in v)

    def run_series(self, n):
        """n steps, observables after every step (device-side series, one copy at the end)."""
        out = {k: np.empty(n, dtype=np.float64) for k in ("E", "M", "M2", "M4")}
        _check(lib().sw_run_series(self._h, int(n), *[out[k].ctypes.data for k in ("E", "M", "M2", "M4")]))
        return out

    def cluster_stats(self):
        """(number of clusters, sum of squared cluster sizes) of the last step's labelling."""
        a, b = C.c_uint64(), C.c_uint64()
        _check(lib().sw_get_cluster_stats(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def counts(self):
        n = self.q if self.model == POTTS else 1
        e = C.c_int64()
        m = (C.c_int64 * n)()
        _check(lib().sw_get_counts(self._h, C.byref(e), m, n))
        return int(e.value), [int(x) for x in m]

    def spins(self, out=None):
        a = out if out is not None else np.empty(self.N, dtype=_SPIN_DTYPE[self.model])
        _check(lib().sw_get_spins(self._h, a.ctypes.data, a.nbytes))
        return a

    def set_spins(self, a, step):
        a = np.ascontiguousarray(a, dtype=_SPIN_DTYPE[self.model])
        _check(lib().sw_set_spins(self._h, a.ctypes.data, a.nbytes, int(step)))

    def get_spins_ptr(self, host_ptr, nbytes):
        _check(lib().sw_get_spins(self._h, C.c_void_p(host_ptr), nbytes))

    def set_spins_ptr(self, host_ptr, nbytes, step):
        _check(lib().sw_set_spins(self._h, C.c_void_p(host_ptr), nbytes, int(step)))

    def bonds(self):
        a = np.empty(self.N, dtype=np.uint8)
        _check(lib().sw_get_bonds(self._h, a.ctypes.data, a.nbytes))
        return a

    def labels(self):
        a = np.empty(self.N, dtype=np.uint32)
        _check(lib().sw_get_labels(self._h, a.ctypes.data, a.nbytes))
        return a

    def clock_hist(self):
        D = np.zeros(self.q, dtype=np.int64)
        n = np.zeros(self.q, dtype=np.int64)
        _check(lib().sw_get_clock_hist(self._h, D.ctypes.data, n.ctypes.data, self.q))
        return D, n

    def clock_mirror(self):
        m = C.c_int()
        _check(lib().sw_get_clock_mirror(self._h, C.byref(m)))
        return int(m.value)

    def xy_dir(self):
        v = [C.c_float() for _ in range(3)]
        _check(lib().sw_get_xy_dir(self._h, *[C.byref(x) for x in v]))
        return tuple(np.float32(x.value) for x in v)

    def force_xy_phi(self, enable, phi=0.0):
        _check(lib().sw_force_xy_phi(self._h, int(bool(enable)), float(phi)))

    def set_counting(self, enable):
        _check(lib().sw_set_counting(self._h, int(bool(enable))))

    def label_stats(self):
        out = (C.c_uint64 * 8)()
        _check(lib().sw_get_label_stats(self._h, out, 8))
        names = ("border_bonds", "active_border_bonds", "unions_linked", "union_retries",
                 "merge_find_hops", "merge_find_hops_max", "chase_hops", "chase_hops_max")
        return dict(zip(names, [int(x) for x in out]))

    def set_kernel_timing(self, enable):
        _check(lib().sw_set_kernel_timing(self._h, int(bool(enable))))

    def kernel_times(self):
        """(ms per kernel [k_bond_label, k_merge, k_flip], steps) accumulated in timing mode."""
        ms = (C.c_double * 3)()
        n = C.c_uint64()
        _check(lib().sw_get_kernel_times(self._h, ms, 3, C.byref(n)))
        return [float(x) for x in ms], int(n.value)
