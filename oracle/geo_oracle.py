"""ctypes binding of the CPU oracle (oracle/geo_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
holds argument marshalling only; every step of the method runs in the C++ file.
It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

SCHWARZSCHILD, KERR = 0, 1
TIMELIKE, NULL = 0, 1
ST_MAXSTEPS, ST_CAPTURED, ST_ESCAPED, ST_NUMERIC = 0, 1, 2, 3
FLAG_PLAIN_UPDATE = 1
FLAG_CARTESIAN_SNAP = 8      # snapshot components r, theta, phi -> x, y, z of eq.(7)


class _Stop(C.Structure):
    _fields_ = [("r_capture", C.c_double), ("r_escape", C.c_double),
                ("kind", C.c_int32), ("flags", C.c_int32)]


class _Out(C.Structure):
    _fields_ = [("final_state", C.c_void_p), ("status", C.c_void_p), ("steps_done", C.c_void_p),
                ("eq_cross_r", C.c_void_p), ("health", C.c_void_p), ("snapshots", C.c_void_p),
                ("snap_capacity", C.c_int64), ("snap_mask", C.c_uint32), ("snap_count", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_integrate.restype = C.c_int
        _lib.oracle_integrate.argtypes = [C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_int64,
                                          C.c_double, C.c_int64, C.POINTER(_Stop), C.c_int64,
                                          C.POINTER(_Out), C.c_int, C.c_int]
        _lib.oracle_rhs.restype = None
        _lib.oracle_rhs.argtypes = [C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_int]
        _lib.oracle_hamiltonian.restype = C.c_double
        _lib.oracle_hamiltonian.argtypes = [C.c_double, C.c_double, C.c_void_p]
        _lib.oracle_energy.restype = C.c_double
        _lib.oracle_energy.argtypes = [C.c_double] * 8
    return _lib


class _Ctl(C.Structure):
    _fields_ = [("h0", C.c_double), ("rtol", C.c_double), ("atol", C.c_double), ("h_min", C.c_double),
                ("tau_end", C.c_double), ("snap_dtau", C.c_double)]


def integrate_adaptive(metric: int, M: float, a: float, state_in: np.ndarray, h0: float, rtol: float,
                       atol: float, max_attempts: int, r_capture: float = -np.inf, r_escape: float = np.inf,
                       kind: int = TIMELIKE, h_min: float = 1e-12, tau_end: float = np.inf,
                       long_double: bool = False, nthreads: int = 1, snap_dtau: float = 0.0,
                       snap_capacity: int = 0, snap_mask: int = 0xFF, flags: int = 0) -> dict:
    """Adaptive Dormand-Prince RK5(4) on host SoA state_in [6][n].  rtol = inf: fixed step h0.
    snap_dtau > 0: dense-output records at tau = j snap_dtau (reading A3), [n][snap_capacity][ncomp]."""
    st = np.ascontiguousarray(state_in, dtype=np.float64)
    n = st.shape[1]
    res = {"final_state": np.full((8, n), np.nan), "status": np.full(n, -1, dtype=np.int32),
           "steps_done": np.zeros(n, dtype=np.int64), "eq_cross_r": np.full(n, np.nan),
           "health": np.full(n, np.nan), "rejected": np.zeros(n, dtype=np.int64), "snapshots": None, "snap_count": None}
    if snap_dtau > 0:
        res["snapshots"] = np.full((n, snap_capacity, bin(snap_mask & 0xFF).count("1")), np.nan)
        res["snap_count"] = np.zeros(n, dtype=np.int32)
    L = lib()
    L.oracle_integrate_adaptive.restype = C.c_int
    L.oracle_integrate_adaptive.argtypes = [C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_int64, C.POINTER(_Ctl),
                                            C.c_int64, C.POINTER(_Stop), C.POINTER(_Out), C.c_void_p, C.c_int, C.c_int]
    stop = _Stop(r_capture, r_escape, kind, flags)
    out = _Out(res["final_state"].ctypes.data, res["status"].ctypes.data, res["steps_done"].ctypes.data,
               res["eq_cross_r"].ctypes.data, res["health"].ctypes.data,
               res["snapshots"].ctypes.data if snap_dtau > 0 else None, snap_capacity, snap_mask,
               res["snap_count"].ctypes.data if snap_dtau > 0 else None)
    ctl = _Ctl(h0, rtol, atol, h_min, tau_end, snap_dtau)
    rc = L.oracle_integrate_adaptive(metric, M, a, st.ctypes.data, n, C.byref(ctl), max_attempts, C.byref(stop),
                                     C.byref(out), res["rejected"].ctypes.data, int(long_double), nthreads)
    if rc != 0:
        raise ValueError("oracle_integrate_adaptive: invalid arguments")
    return res


def dp45_dense_weights(theta: float) -> np.ndarray:
    """w_i(theta), i = 1..7: y(tau_n + theta h) = y_n + h sum_i w_i k_i (reading A3)."""
    w = np.zeros(7)
    L = lib()
    L.oracle_dp45_dense_weights.restype = None
    L.oracle_dp45_dense_weights.argtypes = [C.c_double, C.c_void_p]
    L.oracle_dp45_dense_weights(theta, w.ctypes.data)
    return w


def dp45_tableau() -> dict:
    c, a, b5, b4 = np.zeros(7), np.zeros((7, 7)), np.zeros(7), np.zeros(7)
    L = lib()
    L.oracle_dp45_tableau.restype = None
    L.oracle_dp45_tableau.argtypes = [C.c_void_p] * 4
    L.oracle_dp45_tableau(c.ctypes.data, a.ctypes.data, b5.ctypes.data, b4.ctypes.data)
    return {"c": c, "a": a, "b5": b5, "b4": b4}


def rhs(metric: int, M: float, a: float, y8, long_double: bool = False) -> np.ndarray:
    """d/dtau of (t, r, theta, phi, p_r, p_theta) at y8 = (t, r, theta, phi, E, p_r, p_theta, L)."""
    y = np.ascontiguousarray(y8, dtype=np.float64)
    d = np.empty(6)
    lib().oracle_rhs(metric, M, a, y.ctypes.data, d.ctypes.data, int(long_double))
    return d


def hamiltonian(M: float, a: float, y8) -> float:
    y = np.ascontiguousarray(y8, dtype=np.float64)
    return lib().oracle_hamiltonian(M, a, y.ctypes.data)


def energy(M, a, r, th, pr, pth, L, kappa) -> float:
    """E from the mass shell 2H = -kappa (eq.(5))."""
    return lib().oracle_energy(M, a, r, th, pr, pth, L, kappa)


def integrate(metric: int, M: float, a: float, state_in: np.ndarray, h: float, nsteps: int,
              r_capture: float = -np.inf, r_escape: float = np.inf, kind: int = TIMELIKE,
              flags: int = 0, snapshot_every: int = 0, snap_capacity: int | None = None,
              snap_mask: int = 0xFF, long_double: bool = False, nthreads: int = 1,
              want_eq_cross: bool = True, want_health: bool = True) -> dict:
    """Run the oracle on host SoA state_in [6][n] = (r, theta, phi, u_r, u_theta, u_phi)."""
    st = np.ascontiguousarray(state_in, dtype=np.float64)
    assert st.ndim == 2 and st.shape[0] == 6
    n = st.shape[1]
    ncomp = bin(snap_mask & 0xFF).count("1")
    if snapshot_every > 0 and snap_capacity is None:
        snap_capacity = 1 + nsteps // snapshot_every
    res = {
        "final_state": np.full((8, n), np.nan),
        "status": np.full(n, -1, dtype=np.int32),
        "steps_done": np.zeros(n, dtype=np.int64),
        "eq_cross_r": np.full(n, np.nan) if want_eq_cross else None,
        "health": np.full(n, np.nan) if want_health else None,
        "snapshots": None, "snap_count": None,
    }
    if snapshot_every > 0:
        res["snapshots"] = np.full((n, snap_capacity, ncomp), np.nan)
        res["snap_count"] = np.zeros(n, dtype=np.int32)

    def p(x):
        return None if x is None else x.ctypes.data

    stop = _Stop(r_capture, r_escape, kind, flags)
    out = _Out(p(res["final_state"]), p(res["status"]), p(res["steps_done"]), p(res["eq_cross_r"]),
               p(res["health"]), p(res["snapshots"]), snap_capacity or 0, snap_mask, p(res["snap_count"]))
    rc = lib().oracle_integrate(metric, M, a, st.ctypes.data, n, h, nsteps, C.byref(stop),
                                snapshot_every, C.byref(out), int(long_double), nthreads)
    if rc != 0:
        raise ValueError("oracle_integrate: invalid arguments")
    return res
