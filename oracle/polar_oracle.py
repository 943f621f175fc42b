"""ctypes loader for oracle/polar_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The C file is the oracle (see its header for the definition and citations); this
module only compiles it with gcc for the machine it runs on and marshals numpy
arrays.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "polar_oracle.c")
_SRC_EXT = os.path.join(_HERE, "polar_oracle_ext.c")      # NEXT-4 variants: softening modes, acceleration
_SRC_3D = os.path.join(_HERE, "cartesian_oracle.c")       # NEXT-2: one 3-D Cartesian mesh level
_LIB = None


def _machine_tag() -> str:
    """The .so is built with -march=native, so key it by the CPU's flag set."""
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    with open(_SRC, "rb") as f:
        src = f.read()
    with open(_SRC_EXT, "rb") as f:
        src += f.read()
    with open(_SRC_3D, "rb") as f:
        src += f.read()
    return hashlib.sha1(flags.encode() + src).hexdigest()[:12]


def lib_path() -> str:
    return os.path.join(_HERE, f"libpolar_oracle.{_machine_tag()}.so")


def build(force: bool = False) -> str:
    """Compile polar_oracle.c (gcc -O3 -march=native -fopenmp). Returns the .so path."""
    path = lib_path()
    if force or not os.path.exists(path):
        tmp = path + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared",
               "-o", tmp, _SRC, _SRC_EXT, _SRC_3D, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, path)
    return path


def _lib():
    global _LIB
    if _LIB is None:
        L = ctypes.CDLL(build())
        d, i, l = ctypes.c_double, ctypes.c_int, ctypes.c_long
        p = ctypes.c_void_p
        L.po_num_threads.restype = i
        L.po_grid.argtypes = [i, i, d, d, p, p, p, p]
        L.po_potential_o0_targets.argtypes = [i, i, d, d, d, p, p, l, p]
        L.po_potential_o0_full.argtypes = [i, i, d, d, d, p, p]
        L.po_potential_o1_rings.argtypes = [i, i, d, d, d, p, p, i, p]
        L.po_potential_o1_full.argtypes = [i, i, d, d, d, p, p]
        L.po3_self_constant.restype = d
        L.po3_potential_targets.argtypes = [i, d, p, p, l, p]
        L.po3_potential_full.argtypes = [i, d, p, p]
        L.po3_potential_targets.restype = i
        L.po3_potential_full.restype = i
        L.po_ext_o0_targets.argtypes = [i, i, d, d, d, i, p, p, l, p, p, p]
        L.po_ext_o1_rings.argtypes = [i, i, d, d, d, i, p, p, i, p, p, p]
        for fn in (L.po_grid, L.po_potential_o0_targets, L.po_potential_o0_full,
                   L.po_potential_o1_rings, L.po_potential_o1_full, L.po_ext_o0_targets, L.po_ext_o1_rings):
            fn.restype = i
        _LIB = L
    return _LIB


def _check(st: int, what: str):
    if st != 0:
        raise RuntimeError(f"oracle {what} failed with status {st}")


def _sigma(sigma, n_r, n_phi):
    a = np.ascontiguousarray(sigma, dtype=np.float64)
    if a.shape != (n_r, n_phi):
        raise ValueError(f"sigma must have shape ({n_r},{n_phi}), got {a.shape}")
    return a


def num_threads() -> int:
    return int(_lib().po_num_threads())


def grid(n_r, n_phi, r_in, r_out):
    """Returns (r[n_r], phi[n_phi], area[n_r], edges[n_r+1])."""
    r = np.empty(n_r); phi = np.empty(n_phi); area = np.empty(n_r); edges = np.empty(n_r + 1)
    _check(_lib().po_grid(n_r, n_phi, r_in, r_out, r.ctypes.data, phi.ctypes.data,
                          area.ctypes.data, edges.ctypes.data), "po_grid")
    return r, phi, area, edges


def potential_o0(n_r, n_phi, r_in, r_out, eps, sigma):
    s = _sigma(sigma, n_r, n_phi)
    out = np.empty((n_r, n_phi))
    _check(_lib().po_potential_o0_full(n_r, n_phi, r_in, r_out, eps, s.ctypes.data,
                                       out.ctypes.data), "po_potential_o0_full")
    return out


def potential_o0_targets(n_r, n_phi, r_in, r_out, eps, sigma, targets):
    """targets: flat indices i*n_phi+j. Returns Phi at those cells."""
    s = _sigma(sigma, n_r, n_phi)
    t = np.ascontiguousarray(targets, dtype=np.int64)
    if t.size and (t.min() < 0 or t.max() >= n_r * n_phi):
        raise ValueError("target index out of range")
    out = np.empty(t.size)
    _check(_lib().po_potential_o0_targets(n_r, n_phi, r_in, r_out, eps, s.ctypes.data,
                                          t.ctypes.data, t.size, out.ctypes.data),
           "po_potential_o0_targets")
    return out


def potential_o1(n_r, n_phi, r_in, r_out, eps, sigma):
    s = _sigma(sigma, n_r, n_phi)
    out = np.empty((n_r, n_phi))
    _check(_lib().po_potential_o1_full(n_r, n_phi, r_in, r_out, eps, s.ctypes.data,
                                       out.ctypes.data), "po_potential_o1_full")
    return out


def potential_o1_rings(n_r, n_phi, r_in, r_out, eps, sigma, rings):
    """rings: target ring indices. Returns Phi[len(rings), n_phi]."""
    s = _sigma(sigma, n_r, n_phi)
    rg = np.ascontiguousarray(rings, dtype=np.int32)
    out = np.empty((rg.size, n_phi))
    _check(_lib().po_potential_o1_rings(n_r, n_phi, r_in, r_out, eps, s.ctypes.data,
                                        rg.ctypes.data, rg.size, out.ctypes.data),
           "po_potential_o1_rings")
    return out


# ------------------------------------------------------------------ NEXT-4 variants (polar_oracle_ext.c)
SOFT_SYMMETRIC, SOFT_FIELD, SOFT_SOURCE = 0, 1, 2


def ext_o0_targets(n_r, n_phi, r_in, r_out, eps, soft, sigma, targets):
    """Definition (readings N1, N2) at flat target indices. Returns (Phi, a_r, a_phi)."""
    s = _sigma(sigma, n_r, n_phi)
    t = np.ascontiguousarray(targets, dtype=np.int64)
    if t.size and (t.min() < 0 or t.max() >= n_r * n_phi):
        raise ValueError("target index out of range")
    out = [np.empty(t.size) for _ in range(3)]
    _check(_lib().po_ext_o0_targets(n_r, n_phi, r_in, r_out, eps, int(soft), s.ctypes.data, t.ctypes.data, t.size,
                                    out[0].ctypes.data, out[1].ctypes.data, out[2].ctypes.data), "po_ext_o0_targets")
    return tuple(out)


def ext_o0(n_r, n_phi, r_in, r_out, eps, soft, sigma):
    """Definition on the whole grid. Returns (Phi, a_r, a_phi), each [n_r][n_phi]."""
    out = ext_o0_targets(n_r, n_phi, r_in, r_out, eps, soft, sigma, np.arange(n_r * n_phi))
    return tuple(x.reshape(n_r, n_phi) for x in out)


def ext_o1_rings(n_r, n_phi, r_in, r_out, eps, soft, sigma, rings):
    """Ring-pair form on target rings. Returns (Phi, a_r, a_phi), each [len(rings)][n_phi]."""
    s = _sigma(sigma, n_r, n_phi)
    rg = np.ascontiguousarray(rings, dtype=np.int32)
    out = [np.empty((rg.size, n_phi)) for _ in range(3)]
    _check(_lib().po_ext_o1_rings(n_r, n_phi, r_in, r_out, eps, int(soft), s.ctypes.data, rg.ctypes.data, rg.size,
                                  out[0].ctypes.data, out[1].ctypes.data, out[2].ctypes.data), "po_ext_o1_rings")
    return tuple(out)


def ext_o1(n_r, n_phi, r_in, r_out, eps, soft, sigma):
    return ext_o1_rings(n_r, n_phi, r_in, r_out, eps, soft, sigma, np.arange(n_r))


# ------------------------------------------------------------------ NEXT-2: 3-D Cartesian mesh (cartesian_oracle.c)
def cart_self_constant() -> float:
    return float(_lib().po3_self_constant())


def cart_potential_targets(n, box, rho, targets):
    """Newtonian potential (readings C1-C4) at flat target indices (z*n + y)*n + x."""
    a = np.ascontiguousarray(rho, dtype=np.float64)
    if a.shape != (n, n, n):
        raise ValueError(f"rho must have shape ({n},{n},{n})")
    t = np.ascontiguousarray(targets, dtype=np.int64)
    if t.size and (t.min() < 0 or t.max() >= n**3):
        raise ValueError("target index out of range")
    out = np.empty(t.size)
    _check(_lib().po3_potential_targets(n, box, a.ctypes.data, t.ctypes.data, t.size, out.ctypes.data), "po3_potential_targets")
    return out


def cart_potential(n, box, rho):
    a = np.ascontiguousarray(rho, dtype=np.float64)
    if a.shape != (n, n, n):
        raise ValueError(f"rho must have shape ({n},{n},{n})")
    out = np.empty((n, n, n))
    _check(_lib().po3_potential_full(n, box, a.ctypes.data, out.ctypes.data), "po3_potential_full")
    return out
