"""Thin ctypes binding over libpolargrav.so -- argument marshalling only.

Same names as include/polargrav.h.  Every step of the numerical path runs in the CUDA
kernels; nothing here computes.  If the library is missing this module raises -- there
is no CPU fallback.  PyTorch (optional) is used by callers only for device memory and
streams: pass `tensor.data_ptr()` / `stream.cuda_stream`.
"""
from __future__ import annotations

import ctypes
import os
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpolargrav.so")

PG_OK = 0
PG_ERR_INVALID_ARG, PG_ERR_UNSUPPORTED, PG_ERR_CUDA, PG_ERR_NOMEM, PG_ERR_STATE = -1, -2, -3, -4, -5
PG_MEM_HOST, PG_MEM_HOST_PINNED, PG_MEM_DEVICE = 0, 1, 2
PG_NUM_KERNELS = 3
PG_STATIC_MAX_N = 2048      # largest grid axis of pg_potential_direct_static (its tables are a fixed array)
PG_OPT_DENSITY_STABLE = 1
PG_OPT_LANES = 2
PG_OPT_FUSED = 3
PG_SOFT_SYMMETRIC, PG_SOFT_FIELD, PG_SOFT_SOURCE = 0, 1, 2
KERNEL_NAMES = ("rows_fwd(a2)", "cols(a3+a4r)", "rows_inv(a4phi)")

# every symbol include/polargrav.h declares
EXPORTS = (
    "pg_create", "pg_create_ex", "pg_set_density", "pg_potential", "pg_potential_direct",
    "pg_potential_direct_rings", "pg_destroy", "pg_grid", "pg_set_stream", "pg_set_option", "pg_synchronize",
    "pg_host_alloc", "pg_host_free", "pg_profile", "pg_kernel_times", "pg_launch_count",
    "pg_algorithmic_bytes", "pg_kernel_algorithmic_bytes", "pg_status_string", "pg_last_error",
    "pg_version", "pg_set_softening", "pg_acceleration", "pg_flush", "pg_potential_direct_static", "pg_potential_series",
    "pg3_create", "pg3_set_density", "pg3_potential", "pg3_synchronize", "pg3_destroy", "pg3_launch_count",
    "pg3_algorithmic_bytes", "pg3_last_error",
    "pg3n_create", "pg3n_set_density", "pg3n_restrict", "pg3n_absorb", "pg3n_solve", "pg3n_add_exterior",
    "pg3n_pack_exterior", "pg3n_potential", "pg3n_synchronize", "pg3n_destroy", "pg3n_launch_count", "pg3n_last_error",
    "pg3n_inbox_export", "pg3n_peer_open", "pg3n_peer_set",
)

_lib = None


class PolargravError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"{status_string(status)} ({status}): {message}")
        self.status = status


def lib():
    """Loads libpolargrav.so (once).  Raises if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} not found: build it with `python -m paper_2409_02294_b200.build` "
                "(nvcc, sm_100a).  There is no CPU fallback.")
        L = ctypes.CDLL(LIB_PATH)
        vp, i, d, l = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_long
        L.pg_create.argtypes = [ctypes.POINTER(vp), i, i, d, d, d]
        L.pg_create_ex.argtypes = [ctypes.POINTER(vp), i, i, d, d, d, i, i, vp]
        L.pg_set_density.argtypes = [vp, vp, i, i]
        L.pg_potential.argtypes = [vp, vp, i, i]
        L.pg_potential_direct.argtypes = [vp, vp, i, i]
        L.pg_potential_series.argtypes = [vp, vp, vp, i, ctypes.c_size_t]
        L.pg_potential_direct_rings.argtypes = [vp, vp, i, i, i]
        L.pg_set_softening.argtypes = [vp, i]
        L.pg_acceleration.argtypes = [vp, vp, vp, i, i]
        L.pg_destroy.argtypes = [vp]
        L.pg_potential_direct_static.argtypes = [vp, vp, i, i, d, d, d, i, vp]
        L.pg_grid.argtypes = [vp, vp, vp, vp]
        L.pg_set_stream.argtypes = [vp, vp]
        L.pg_set_option.argtypes = [vp, i, i]
        L.pg_synchronize.argtypes = [vp]
        L.pg_flush.argtypes = [vp]
        L.pg_host_alloc.argtypes = [ctypes.POINTER(vp), ctypes.c_size_t]
        L.pg_host_free.argtypes = [vp]
        L.pg_profile.argtypes = [vp, i]
        L.pg_kernel_times.argtypes = [vp, ctypes.POINTER(d), ctypes.POINTER(l)]
        L.pg3_create.argtypes = [ctypes.POINTER(vp), i, d, i, vp]
        L.pg3_set_density.argtypes = [vp, vp, i]
        L.pg3_potential.argtypes = [vp, vp, i]
        L.pg3_synchronize.argtypes = [vp]
        L.pg3_destroy.argtypes = [vp]
        L.pg3n_create.argtypes = [ctypes.POINTER(vp), i, d, i, i, i, vp]
        L.pg3n_set_density.argtypes = [vp, vp, i]
        L.pg3n_restrict.argtypes = [vp, vp]
        L.pg3n_absorb.argtypes = [vp, vp]
        L.pg3n_solve.argtypes = [vp]
        L.pg3n_add_exterior.argtypes = [vp, vp]
        L.pg3n_pack_exterior.argtypes = [vp, vp]
        L.pg3n_potential.argtypes = [vp, vp, i]
        L.pg3n_synchronize.argtypes = [vp]
        L.pg3n_destroy.argtypes = [vp]
        L.pg3n_inbox_export.argtypes = [vp, i, ctypes.c_char_p, ctypes.POINTER(vp)]
        L.pg3n_peer_open.argtypes = [vp, i, ctypes.c_char_p]
        L.pg3n_peer_set.argtypes = [vp, i, vp]
        for name in EXPORTS:
            getattr(L, name).restype = i
        L.pg3n_launch_count.argtypes = [vp]; L.pg3n_launch_count.restype = l
        L.pg3n_last_error.argtypes = [vp]; L.pg3n_last_error.restype = ctypes.c_char_p
        L.pg3_launch_count.argtypes = [vp]; L.pg3_launch_count.restype = l
        L.pg3_algorithmic_bytes.argtypes = [vp]; L.pg3_algorithmic_bytes.restype = d
        L.pg3_last_error.argtypes = [vp]; L.pg3_last_error.restype = ctypes.c_char_p
        L.pg_launch_count.argtypes = [vp]; L.pg_launch_count.restype = l
        L.pg_algorithmic_bytes.argtypes = [vp, i]; L.pg_algorithmic_bytes.restype = d
        L.pg_kernel_algorithmic_bytes.argtypes = [vp, i, i]; L.pg_kernel_algorithmic_bytes.restype = d
        L.pg_status_string.argtypes = [i]; L.pg_status_string.restype = ctypes.c_char_p
        L.pg_last_error.argtypes = [vp]; L.pg_last_error.restype = ctypes.c_char_p
        L.pg_version.argtypes = []; L.pg_version.restype = ctypes.c_char_p
        _lib = L
    return _lib


def status_string(st: int) -> str:
    return lib().pg_status_string(int(st)).decode()


def last_error(handle=None) -> str:
    return lib().pg_last_error(handle).decode()


def version() -> str:
    return lib().pg_version().decode()


def _check(st, handle=None):
    if st != PG_OK:
        raise PolargravError(st, last_error(handle))


def _ptr(x):
    """Address of a numpy array / int address / object with data_ptr() (torch tensor)."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        if x.dtype != np.float64 or not x.flags.c_contiguous:
            raise TypeError("arrays must be C-contiguous float64")
        return x.ctypes.data
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    return int(x)


# ------------------------------------------------------------------ the C ABI, same names
def pg_create(n_r, n_phi, r_in, r_out, eps):
    h = ctypes.c_void_p()
    st = lib().pg_create(ctypes.byref(h), n_r, n_phi, r_in, r_out, eps)
    _check(st)
    return h


def pg_create_ex(n_r, n_phi, r_in, r_out, eps, max_batch=1, device=-1, cuda_stream=None):
    h = ctypes.c_void_p()
    st = lib().pg_create_ex(ctypes.byref(h), n_r, n_phi, r_in, r_out, eps, max_batch, device,
                            ctypes.c_void_p(cuda_stream) if cuda_stream else None)
    _check(st)
    return h


def pg_set_density(h, sigma, batch, where):
    _check(lib().pg_set_density(h, _ptr(sigma), batch, where), h)


def pg_potential(h, phi, batch, where):
    _check(lib().pg_potential(h, _ptr(phi), batch, where), h)


def pg_potential_series(h, sigma, phi, count, stride):
    _check(lib().pg_potential_series(h, _ptr(sigma), _ptr(phi), count, stride), h)


def pg_potential_direct(h, phi, batch, where):
    _check(lib().pg_potential_direct(h, _ptr(phi), batch, where), h)


def pg_potential_direct_rings(h, phi, ring0, n_rings, where):
    _check(lib().pg_potential_direct_rings(h, _ptr(phi), ring0, n_rings, where), h)


def pg_set_softening(h, mode):
    _check(lib().pg_set_softening(h, int(mode)), h)


def pg_acceleration(h, a_r, a_phi, batch, where):
    _check(lib().pg_acceleration(h, _ptr(a_r), _ptr(a_phi), batch, where), h)


def pg_destroy(h):
    _check(lib().pg_destroy(h))


def pg_potential_direct_static(sigma, phi, n_r, n_phi, r_in, r_out, eps, device=-1, cuda_stream=None):
    """Direct summation of one field with no solver and no allocation (tables in a fixed 48 KiB array of the library);
    sigma, phi: device arrays.  Errors carry the text of pg_last_error(NULL)."""
    _check(lib().pg_potential_direct_static(_ptr(sigma), _ptr(phi), n_r, n_phi, r_in, r_out, eps, device,
                                            ctypes.c_void_p(cuda_stream) if cuda_stream else None))


def pg_grid(h, n_r, n_phi):
    r, phi, area = np.empty(n_r), np.empty(n_phi), np.empty(n_r)
    _check(lib().pg_grid(h, r.ctypes.data, phi.ctypes.data, area.ctypes.data), h)
    return r, phi, area


def pg_set_stream(h, cuda_stream):
    _check(lib().pg_set_stream(h, ctypes.c_void_p(cuda_stream) if cuda_stream else None), h)


def pg_set_option(h, option, value):
    _check(lib().pg_set_option(h, int(option), int(value)), h)


def pg_flush(h):
    _check(lib().pg_flush(h), h)


def pg_synchronize(h):
    _check(lib().pg_synchronize(h), h)


def pg_host_alloc(nbytes):
    p = ctypes.c_void_p()
    _check(lib().pg_host_alloc(ctypes.byref(p), nbytes))
    return p.value


def pg_host_free(p):
    _check(lib().pg_host_free(ctypes.c_void_p(p)))


def pg_profile(h, enable):
    _check(lib().pg_profile(h, int(bool(enable))), h)


def pg_kernel_times(h):
    ms = (ctypes.c_double * PG_NUM_KERNELS)()
    n = (ctypes.c_long * PG_NUM_KERNELS)()
    _check(lib().pg_kernel_times(h, ms, n), h)
    return list(ms), list(n)


def pg_launch_count(h):
    return int(lib().pg_launch_count(h))


def pg_algorithmic_bytes(h, batch=1):
    return float(lib().pg_algorithmic_bytes(h, batch))


def pg_kernel_algorithmic_bytes(h, index, batch=1):
    return float(lib().pg_kernel_algorithmic_bytes(h, index, batch))


# ------------------------------------------------------------------ NEXT-2: 3-D Cartesian mesh level
def _check3(st, handle=None):
    if st != PG_OK:
        msg = lib().pg3_last_error(handle).decode()
        raise PolargravError(st, f"{status_string(st)}: {msg}")


def pg3_create(n, box, device=-1, cuda_stream=None):
    h = ctypes.c_void_p()
    _check3(lib().pg3_create(ctypes.byref(h), n, box, device, ctypes.c_void_p(cuda_stream) if cuda_stream else None))
    return h


def pg3_set_density(h, rho, where):
    _check3(lib().pg3_set_density(h, _ptr(rho), where), h)


def pg3_potential(h, phi, where):
    _check3(lib().pg3_potential(h, _ptr(phi), where), h)


def pg3_synchronize(h):
    _check3(lib().pg3_synchronize(h), h)


def pg3_destroy(h):
    _check3(lib().pg3_destroy(h))


def pg3_launch_count(h):
    return int(lib().pg3_launch_count(h))


def pg3_algorithmic_bytes(h):
    return float(lib().pg3_algorithmic_bytes(h))


def pg3_last_error(h=None):
    return lib().pg3_last_error(h).decode()


# ------------------------------------------------------------------ NEXT-3: nested 3-D mesh levels
def _check3n(st, handle=None):
    if st != PG_OK:
        msg = lib().pg3n_last_error(handle).decode()
        raise PolargravError(st, f"{status_string(st)}: {msg}")


def pg3n_create(n, box0, level, depth, device=-1, cuda_stream=None):
    h = ctypes.c_void_p()
    _check3n(lib().pg3n_create(ctypes.byref(h), n, box0, level, depth, device,
                               ctypes.c_void_p(cuda_stream) if cuda_stream else None))
    return h


def pg3n_set_density(h, rho, where):
    _check3n(lib().pg3n_set_density(h, _ptr(rho), where), h)


def pg3n_restrict(h, child_mean_out):
    _check3n(lib().pg3n_restrict(h, _ptr(child_mean_out)), h)


def pg3n_absorb(h, child_mean):
    _check3n(lib().pg3n_absorb(h, _ptr(child_mean)), h)


def pg3n_solve(h):
    _check3n(lib().pg3n_solve(h), h)


def pg3n_add_exterior(h, parent_halo):
    _check3n(lib().pg3n_add_exterior(h, _ptr(parent_halo)), h)


def pg3n_pack_exterior(h, halo_out):
    _check3n(lib().pg3n_pack_exterior(h, _ptr(halo_out)), h)


def pg3n_potential(h, phi, where):
    _check3n(lib().pg3n_potential(h, _ptr(phi), where), h)


def pg3n_synchronize(h):
    _check3n(lib().pg3n_synchronize(h), h)


def pg3n_destroy(h):
    _check3n(lib().pg3n_destroy(h))


PG3N_INBOX_MEAN, PG3N_INBOX_HALO = 0, 1
PG_IPC_HANDLE_BYTES = 64


def pg3n_inbox_export(h, which):
    """(IPC handle as 64 bytes, device address) of this level's inbox `which`; allocates it on first use."""
    buf = ctypes.create_string_buffer(PG_IPC_HANDLE_BYTES)
    ptr = ctypes.c_void_p()
    _check3n(lib().pg3n_inbox_export(h, which, buf, ctypes.byref(ptr)), h)
    return buf.raw, ptr.value


def pg3n_peer_open(h, which, handle: bytes):
    if len(handle) != PG_IPC_HANDLE_BYTES:
        raise ValueError("an IPC handle has 64 bytes")
    _check3n(lib().pg3n_peer_open(h, which, handle), h)


def pg3n_peer_set(h, which, device_address):
    _check3n(lib().pg3n_peer_set(h, which, device_address), h)


def pg3n_launch_count(h):
    return int(lib().pg3n_launch_count(h))


def pg3n_last_error(h=None):
    return lib().pg3n_last_error(h).decode()


# ------------------------------------------------------------------ convenience wrapper
class PinnedArray:
    """float64 numpy view over page-locked memory owned by the CUDA side (pg_host_alloc)."""

    def __init__(self, shape):
        self.shape = tuple(shape)
        n = int(np.prod(self.shape))
        self.ptr = pg_host_alloc(n * 8)
        buf = (ctypes.c_double * n).from_address(self.ptr)
        self.array = np.frombuffer(buf, dtype=np.float64).reshape(self.shape)

    def free(self):
        if self.ptr:
            self.array = None
            pg_host_free(self.ptr)
            self.ptr = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Solver:
    """RAII wrapper; methods marshal arguments and call the C ABI, nothing else."""

    def __init__(self, n_r, n_phi, r_in, r_out, eps, max_batch=1, device=-1, cuda_stream=None):
        self.n_r, self.n_phi, self.max_batch = n_r, n_phi, max_batch
        self.h = pg_create_ex(n_r, n_phi, r_in, r_out, eps, max_batch, device, cuda_stream)

    def grid(self):
        return pg_grid(self.h, self.n_r, self.n_phi)

    def potential_host(self, sigma: np.ndarray, direct: bool = False) -> np.ndarray:
        """Host numpy in, host numpy out (pageable path, PG_MEM_HOST)."""
        s = np.ascontiguousarray(sigma, dtype=np.float64)
        batch = 1 if s.ndim == 2 else s.shape[0]
        if s.shape[-2:] != (self.n_r, self.n_phi):
            raise ValueError("sigma has the wrong shape")
        out = np.empty_like(s)
        pg_set_density(self.h, s, batch, PG_MEM_HOST)
        (pg_potential_direct if direct else pg_potential)(self.h, out, batch, PG_MEM_HOST)
        return out

    def close(self):
        if self.h is not None:
            pg_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
