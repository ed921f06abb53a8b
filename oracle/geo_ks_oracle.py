"""ctypes binding of the Cartesian Kerr-Schild CPU oracle (oracle/geo_ks_oracle.cpp, readings K1-K5).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import
this module.  Argument marshalling only; it imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

TIMELIKE, NULL = 0, 1
ST_MAXSTEPS, ST_CAPTURED, ST_ESCAPED, ST_NUMERIC = 0, 1, 2, 3
FLAG_PLAIN_UPDATE = 1


class _Stop(C.Structure):
    _fields_ = [("r_capture", C.c_double), ("r_escape", C.c_double), ("kind", C.c_int32), ("flags", C.c_int32)]


class _Out(C.Structure):
    _fields_ = [("final_state", C.c_void_p), ("status", C.c_void_p), ("steps_done", C.c_void_p),
                ("eq_cross_r", C.c_void_p), ("health", C.c_void_p), ("snapshots", C.c_void_p),
                ("snap_capacity", C.c_int64), ("snap_mask", C.c_uint32), ("snap_count", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_ks_integrate.restype = C.c_int
        _lib.oracle_ks_integrate.argtypes = [C.c_double, C.c_double, C.c_void_p, C.c_int64, C.c_double, C.c_int64,
                                             C.POINTER(_Stop), C.c_int64, C.POINTER(_Out), C.c_int, C.c_int]
        _lib.oracle_ks_rhs.restype = None
        _lib.oracle_ks_rhs.argtypes = [C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_int]
        _lib.oracle_ks_hamiltonian.restype = C.c_double
        _lib.oracle_ks_hamiltonian.argtypes = [C.c_double, C.c_double, C.c_void_p]
        _lib.oracle_ks_energy.restype = C.c_double
        _lib.oracle_ks_energy.argtypes = [C.c_double] * 9
        _lib.oracle_ks_radius.restype = C.c_double
        _lib.oracle_ks_radius.argtypes = [C.c_double] * 5
        _lib.oracle_ks_metric.restype = None
        _lib.oracle_ks_metric.argtypes = [C.c_double] * 5 + [C.c_void_p]
    return _lib


def rhs(M: float, a: float, y8, long_double: bool = False) -> np.ndarray:
    """d/dtau of (t~, x, y, z, p_x, p_y, p_z) at y8 = (t~, x, y, z, E, p_x, p_y, p_z)."""
    y = np.ascontiguousarray(y8, dtype=np.float64)
    d = np.empty(7)
    lib().oracle_ks_rhs(M, a, y.ctypes.data, d.ctypes.data, int(long_double))
    return d


def hamiltonian(M: float, a: float, y8) -> float:
    y = np.ascontiguousarray(y8, dtype=np.float64)
    return lib().oracle_ks_hamiltonian(M, a, y.ctypes.data)


def energy(M, a, x, y, z, px, py, pz, kappa) -> float:
    """E from the mass shell 2H = -kappa in 3+1 variables (eq.(5))."""
    return lib().oracle_ks_energy(M, a, x, y, z, px, py, pz, kappa)


def radius(M, a, x, y, z) -> float:
    return lib().oracle_ks_radius(M, a, x, y, z)


def metric(M, a, x, y, z) -> np.ndarray:
    """(f, l_x, l_y, l_z) of g = eta + f l l at a point."""
    o = np.empty(4)
    lib().oracle_ks_metric(M, a, x, y, z, o.ctypes.data)
    return o


def integrate(M: float, a: float, state_in: np.ndarray, h: float, nsteps: int, r_capture: float = -np.inf,
              r_escape: float = np.inf, kind: int = TIMELIKE, flags: int = 0, snapshot_every: int = 0,
              snap_capacity: int | None = None, snap_mask: int = 0xFF, long_double: bool = False,
              nthreads: int = 1) -> dict:
    """Run the oracle on host SoA state_in [6][n] = (x, y, z, p_x, p_y, p_z)."""
    st = np.ascontiguousarray(state_in, dtype=np.float64)
    assert st.ndim == 2 and st.shape[0] == 6
    n = st.shape[1]
    ncomp = bin(snap_mask & 0xFF).count("1")
    res = {"final_state": np.full((8, n), np.nan), "status": np.full(n, -1, dtype=np.int32),
           "steps_done": np.zeros(n, dtype=np.int64), "eq_cross_r": np.full(n, np.nan),
           "health": np.full(n, np.nan), "snapshots": None, "snap_count": None}
    if snapshot_every > 0:
        if snap_capacity is None:
            snap_capacity = 1 + nsteps // snapshot_every
        res["snapshots"] = np.full((n, snap_capacity, ncomp), np.nan)
        res["snap_count"] = np.zeros(n, dtype=np.int32)
    stop = _Stop(r_capture, r_escape, kind, flags)
    out = _Out(res["final_state"].ctypes.data, res["status"].ctypes.data, res["steps_done"].ctypes.data,
               res["eq_cross_r"].ctypes.data, res["health"].ctypes.data,
               res["snapshots"].ctypes.data if snapshot_every > 0 else None, snap_capacity or 0, snap_mask,
               res["snap_count"].ctypes.data if snapshot_every > 0 else None)
    rc = lib().oracle_ks_integrate(M, a, st.ctypes.data, n, h, nsteps, C.byref(stop), snapshot_every, C.byref(out),
                                   int(long_double), nthreads)
    if rc != 0:
        raise ValueError("oracle_ks_integrate: invalid arguments")
    return res


class _Ctl(C.Structure):
    _fields_ = [("h0", C.c_double), ("rtol", C.c_double), ("atol", C.c_double), ("h_min", C.c_double),
                ("tau_end", C.c_double), ("snap_dtau", C.c_double)]


def integrate_adaptive(M: float, a: float, state_in: np.ndarray, h0: float, rtol: float, atol: float, max_attempts: int,
                       r_capture: float = -np.inf, r_escape: float = np.inf, kind: int = TIMELIKE, h_min: float = 1e-12,
                       tau_end: float = np.inf, long_double: bool = False, nthreads: int = 1, snap_dtau: float = 0.0,
                       snap_capacity: int = 0, snap_mask: int = 0xFF) -> dict:
    """Adaptive Dormand-Prince RK5(4) in the Kerr-Schild chart (reading K6) on host SoA state_in [6][n]; rtol = inf: fixed step."""
    st = np.ascontiguousarray(state_in, dtype=np.float64)
    n = st.shape[1]
    res = {"final_state": np.full((8, n), np.nan), "status": np.full(n, -1, dtype=np.int32),
           "steps_done": np.zeros(n, dtype=np.int64), "eq_cross_r": np.full(n, np.nan), "health": np.full(n, np.nan),
           "rejected": np.zeros(n, dtype=np.int64), "snapshots": None, "snap_count": None}
    if snap_dtau > 0:
        res["snapshots"] = np.full((n, snap_capacity, bin(snap_mask & 0xFF).count("1")), np.nan)
        res["snap_count"] = np.zeros(n, dtype=np.int32)
    stop = _Stop(r_capture, r_escape, kind, 0)
    out = _Out(res["final_state"].ctypes.data, res["status"].ctypes.data, res["steps_done"].ctypes.data,
               res["eq_cross_r"].ctypes.data, res["health"].ctypes.data,
               res["snapshots"].ctypes.data if snap_dtau > 0 else None, snap_capacity, snap_mask,
               res["snap_count"].ctypes.data if snap_dtau > 0 else None)
    ctl = _Ctl(h0, rtol, atol, h_min, tau_end, snap_dtau)
    L = lib()
    L.oracle_ks_integrate_adaptive.restype = C.c_int
    L.oracle_ks_integrate_adaptive.argtypes = [C.c_double, C.c_double, C.c_void_p, C.c_int64, C.POINTER(_Ctl), C.c_int64,
                                               C.POINTER(_Stop), C.POINTER(_Out), C.c_void_p, C.c_int, C.c_int]
    rc = L.oracle_ks_integrate_adaptive(M, a, st.ctypes.data, n, C.byref(ctl), max_attempts, C.byref(stop), C.byref(out),
                                        res["rejected"].ctypes.data, int(long_double), nthreads)
    if rc != 0:
        raise ValueError("oracle_ks_integrate_adaptive: invalid arguments")
    return res
