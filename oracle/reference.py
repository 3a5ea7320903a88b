"""ctypes front-end of oracle/sg_oracle.c (TEST INFRASTRUCTURE; see that file's header)."""
from __future__ import annotations

import ctypes
import numpy as np

from .build import build

_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        i64p = ctypes.POINTER(ctypes.c_int64)
        f64p = ctypes.POINTER(ctypes.c_double)
        for sfx in ("f80", "f64"):
            f = getattr(_lib, f"sg_oracle_force_{sfx}")
            f.restype = ctypes.c_int
            f.argtypes = [ctypes.c_int64, i64p, i64p, i64p, i64p, f64p, f64p, f64p,
                          ctypes.c_int64, i64p, i64p, ctypes.c_double, ctypes.c_double, f64p, f64p,
                          ctypes.c_int]
            k = getattr(_lib, f"sg_oracle_cell_kernels_{sfx}")
            k.restype = None
            k.argtypes = [ctypes.c_int64] * 6 + [ctypes.c_double, f64p]
    return _lib


def _i64(a):
    a = np.ascontiguousarray(a, dtype=np.int64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


def _f64(a):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def force(rects, sigma, ktx, kty, unit, G=1.0, dx=None, dy=None, precision="f80", n_threads=0):
    """Fx, Fy at integer-lattice targets (ktx, kty) from the leaf rectangles ``rects``
    (dict with int64 kxl, kxr, kyd, kyu as produced by workloads.cell_rects).

    Returns (Fx, Fy, threads_used).  precision: "f80" (long double) or "f64".
    """
    lib = _load()
    a1, p1 = _i64(rects["kxl"]); a2, p2 = _i64(rects["kxr"])
    a3, p3 = _i64(rects["kyd"]); a4, p4 = _i64(rects["kyu"])
    s, ps = _f64(sigma)
    d1, pd1 = _f64(dx); d2, pd2 = _f64(dy)
    tx, ptx = _i64(ktx); ty, pty = _i64(kty)
    n_t = tx.size
    Fx = np.empty(n_t); Fy = np.empty(n_t)
    fn = getattr(lib, f"sg_oracle_force_{precision}")
    used = fn(a1.size, p1, p2, p3, p4, ps, pd1, pd2, n_t, ptx, pty, float(unit), float(G),
              Fx.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
              Fy.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(n_threads))
    return Fx, Fy, used


def cell_kernels(kxl, kxr, kyd, kyu, ktx, kty, unit, precision="f80"):
    """(Kx0, Kxx, Kxy, Ky0, Kyx, Kyy) of one rectangle at one target (z = 0)."""
    lib = _load()
    out = np.empty(6)
    getattr(lib, f"sg_oracle_cell_kernels_{precision}")(
        int(kxl), int(kxr), int(kyd), int(kyu), int(ktx), int(kty), float(unit),
        out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return out
