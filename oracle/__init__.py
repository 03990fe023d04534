"""ctypes binding of the CPU oracle (oracle/swept_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference` legs may
import this package.  It shares nothing with the CUDA path (`paper_1612_02495_b200/`).

Each function advances a copy of the given field by `nsteps` naive timesteps on the periodic grid,
in the dtype of the array it is given (float32 or float64), and returns the new array.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import build as _build

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        for suf, ptr in (("f64", ctypes.POINTER(ctypes.c_double)), ("f32", ctypes.POINTER(ctypes.c_float))):
            f = getattr(L, f"oracle_heat_{suf}")
            f.argtypes = [ptr, ctypes.c_long, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double]
            f.restype = ctypes.c_int
            f = getattr(L, f"oracle_heat_insulated_{suf}")
            f.argtypes = [ptr, ctypes.c_long, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double]
            f.restype = ctypes.c_int
            f = getattr(L, f"oracle_heat2d_{suf}")
            f.argtypes = [ptr, ctypes.c_long, ctypes.c_long, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double]
            f.restype = ctypes.c_int
            f = getattr(L, f"oracle_ks_{suf}")
            f.argtypes = [ptr, ctypes.c_long, ctypes.c_long, ctypes.c_double, ctypes.c_double]
            f.restype = ctypes.c_int
            f = getattr(L, f"oracle_euler_{suf}")
            f.argtypes = [ptr, ctypes.c_long, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double]
            f.restype = ctypes.c_int
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


def _prep(u: np.ndarray, ncomp: int):
    if u.dtype not in (np.float32, np.float64):
        raise TypeError("oracle runs in float32 or float64 only")
    a = np.array(u, copy=True, order="C")
    flat = a.reshape(-1)
    if ncomp == 1:
        nx = flat.size
    else:
        if a.ndim != 2 or a.shape[0] != ncomp:
            raise ValueError(f"expected shape [{ncomp}, nx]")
        nx = a.shape[1]
    suf = "f64" if a.dtype == np.float64 else "f32"
    cty = ctypes.c_double if a.dtype == np.float64 else ctypes.c_float
    return a, flat.ctypes.data_as(ctypes.POINTER(cty)), nx, suf


def heat(u: np.ndarray, nsteps: int, alpha: float, dx: float, dt: float) -> np.ndarray:
    """FTCS heat, Eq. (2), periodic."""
    a, p, nx, suf = _prep(u, 1)
    rc = getattr(lib(), f"oracle_heat_{suf}")(p, nx, int(nsteps), float(alpha), float(dx), float(dt))
    if rc != 0:
        raise RuntimeError(f"oracle_heat failed rc={rc}")
    return a


def heat_insulated(u: np.ndarray, nsteps: int, alpha: float, dx: float, dt: float) -> np.ndarray:
    """FTCS heat on a rod with insulated ends (Eq. 9, reading G7: ghost = adjacent interior value)."""
    a, p, nx, suf = _prep(u, 1)
    rc = getattr(lib(), f"oracle_heat_insulated_{suf}")(p, nx, int(nsteps), float(alpha), float(dx), float(dt))
    if rc != 0:
        raise RuntimeError(f"oracle_heat_insulated failed rc={rc}")
    return a


def heat2d(u: np.ndarray, nsteps: int, alpha: float, dx: float, dt: float) -> np.ndarray:
    """2-D FTCS heat (5-point), periodic in both directions; u has shape [ny, nx] (row-major, x fastest)."""
    if u.dtype not in (np.float32, np.float64) or u.ndim != 2:
        raise TypeError("oracle.heat2d takes a 2-D float32 / float64 array [ny, nx]")
    a = np.array(u, copy=True, order="C")
    suf = "f64" if a.dtype == np.float64 else "f32"
    cty = ctypes.c_double if a.dtype == np.float64 else ctypes.c_float
    rc = getattr(lib(), f"oracle_heat2d_{suf}")(a.ctypes.data_as(ctypes.POINTER(cty)), a.shape[1], a.shape[0], int(nsteps), float(alpha), float(dx), float(dt))
    if rc != 0:
        raise RuntimeError(f"oracle_heat2d failed rc={rc}")
    return a


def ks(u: np.ndarray, nsteps: int, dx: float, dt: float) -> np.ndarray:
    """Kuramoto-Sivashinsky, Eq. (4) + (15) + (16) PAPER.md:64, 291, 295, periodic."""
    a, p, nx, suf = _prep(u, 1)
    rc = getattr(lib(), f"oracle_ks_{suf}")(p, nx, int(nsteps), float(dx), float(dt))
    if rc != 0:
        raise RuntimeError(f"oracle_ks failed rc={rc}")
    return a


def euler(U: np.ndarray, nsteps: int, gamma: float, dx: float, dt: float, check_positive: bool = True) -> np.ndarray:
    """Euler MUSCL/minmod/Rusanov midpoint (BASELINE.json config 4), U = [rho, m, E] rows, periodic."""
    a, p, nx, suf = _prep(U, 3)
    rc = getattr(lib(), f"oracle_euler_{suf}")(p, nx, int(nsteps), float(gamma), float(dx), float(dt))
    if rc < 0:
        raise RuntimeError(f"oracle_euler failed rc={rc}")
    if rc == 1 and check_positive:
        raise FloatingPointError("oracle_euler: density or pressure became non-positive (reading E4)")
    return a


def run(problem: int, u: np.ndarray, nsteps: int, *, dx: float, dt: float, alpha: float = 1.0, gamma: float = 1.4,
        insulated: bool = False) -> np.ndarray:
    """Dispatch on the problem id (0 heat, 1 KS, 2 Euler); arrays are [ncomp, nx]."""
    if problem == 0:
        return heat_insulated(u, nsteps, alpha, dx, dt) if insulated else heat(u, nsteps, alpha, dx, dt)
    if problem == 1:
        return ks(u, nsteps, dx, dt)
    if problem == 2:
        return euler(u, nsteps, gamma, dx, dt)
    raise ValueError(f"unknown problem {problem}")


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))
