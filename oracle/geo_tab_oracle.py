"""ctypes binding of the tabulated-metric CPU oracle (oracle/geo_tab_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  Argument marshalling only; imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

TIMELIKE, NULL = 0, 1
ST_MAXSTEPS, ST_CAPTURED, ST_ESCAPED, ST_NUMERIC, ST_OUTSIDE = 0, 1, 2, 3, 4


class _Stop(C.Structure):
    _fields_ = [("r_capture", C.c_double), ("r_escape", C.c_double), ("kind", C.c_int32), ("flags", C.c_int32)]


class _Out(C.Structure):
    _fields_ = [("final_state", C.c_void_p), ("status", C.c_void_p), ("steps_done", C.c_void_p),
                ("eq_cross_r", C.c_void_p), ("health", C.c_void_p), ("snapshots", C.c_void_p),
                ("snap_capacity", C.c_int64), ("snap_mask", C.c_uint32), ("snap_count", C.c_void_p)]


_lib = None
_GRID = [C.c_void_p, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_tab_integrate.restype = C.c_int
        _lib.oracle_tab_integrate.argtypes = _GRID + [C.c_void_p, C.c_int64, C.c_double, C.c_int64, C.POINTER(_Stop),
                                                      C.POINTER(_Out), C.c_int, C.c_int, C.c_int64]
        _lib.oracle_tab_fields.restype = C.c_int
        _lib.oracle_tab_fields.argtypes = _GRID + [C.c_double, C.c_double, C.c_void_p]
        _lib.oracle_tab_rhs.restype = C.c_int
        _lib.oracle_tab_rhs.argtypes = _GRID + [C.c_void_p, C.c_void_p, C.c_void_p]
    return _lib


def _grid(table: dict, nf: int = 5):
    tab = table["tab"]
    assert tab.dtype == np.float64 and tab.flags.c_contiguous and tab.ndim == 3 and tab.shape[0] == nf
    return [tab.ctypes.data, tab.shape[2], tab.shape[1], table["x1_0"], table["d1"], table["x2_0"], table["d2"]]


def fields(table: dict, x1: float, x2: float):
    """(value[5], d/dx1[5], d/dx2[5]) of the interpolated alpha, beta^phi, gamma_11, gamma_22, gamma_33; None outside."""
    out = np.zeros(15)
    ok = lib().oracle_tab_fields(*_grid(table), x1, x2, out.ctypes.data)
    return (out[:5], out[5:10], out[10:]) if ok else None


def rhs(table: dict, y8):
    """d/dtau of (t, x1, x2, phi, p1, p2) and H at y8 = (t, x1, x2, phi, E, p1, p2, L); None outside the domain."""
    y = np.ascontiguousarray(y8, dtype=np.float64)
    d, H = np.zeros(6), C.c_double()
    ok = lib().oracle_tab_rhs(*_grid(table), y.ctypes.data, d.ctypes.data, C.byref(H))
    return (d, H.value) if ok else None


def integrate(table: dict, state_in: np.ndarray, h: float, nsteps: int, r_capture: float = -np.inf,
              r_escape: float = np.inf, kind: int = TIMELIKE, flags: int = 0, long_double: bool = False,
              nthreads: int = 1, snapshot_every: int = 0, snap_capacity: int | None = None, snap_mask: int = 0xFF) -> dict:
    """Fixed-step RK4 through the tabulated metric on host SoA state_in [6][n] = (x1, x2, phi, p_1, p_2, p_phi)."""
    st = np.ascontiguousarray(state_in, dtype=np.float64)
    n = st.shape[1]
    res = {"final_state": np.full((8, n), np.nan), "status": np.full(n, -1, dtype=np.int32),
           "steps_done": np.zeros(n, dtype=np.int64), "eq_cross_r": np.full(n, np.nan), "health": np.full(n, np.nan),
           "snapshots": None, "snap_count": None}
    if snapshot_every > 0:
        if snap_capacity is None:
            snap_capacity = 1 + nsteps // snapshot_every
        res["snapshots"] = np.full((n, snap_capacity, bin(snap_mask & 0xFF).count("1")), np.nan)
        res["snap_count"] = np.zeros(n, dtype=np.int32)
    stop = _Stop(r_capture, r_escape, kind, flags)
    out = _Out(res["final_state"].ctypes.data, res["status"].ctypes.data, res["steps_done"].ctypes.data,
               res["eq_cross_r"].ctypes.data, res["health"].ctypes.data,
               res["snapshots"].ctypes.data if snapshot_every > 0 else None, snap_capacity or 0, snap_mask,
               res["snap_count"].ctypes.data if snapshot_every > 0 else None)
    rc = lib().oracle_tab_integrate(*_grid(table), st.ctypes.data, n, h, nsteps, C.byref(stop), C.byref(out),
                                    int(long_double), nthreads, snapshot_every)
    if rc != 0:
        raise ValueError("oracle_tab_integrate: invalid arguments")
    return res


# ---- reading T6: general stationary axisymmetric 3+1 metric, tab [10][n2][n1] =
#      alpha, beta^1, beta^2, beta^3, gamma_11, gamma_12, gamma_13, gamma_22, gamma_23, gamma_33 ----
def rhs_general(table: dict, y8, kappa: float = 1.0):
    """(d/dtau of (t, x1, x2, phi, p1, p2), H, mass-shell E) at y8 = (t, x1, x2, phi, E, p1, p2, L); None outside."""
    y = np.ascontiguousarray(y8, dtype=np.float64)
    d, H, E = np.zeros(6), C.c_double(), C.c_double()
    L = lib()
    L.oracle_tabg_rhs.restype = C.c_int
    L.oracle_tabg_rhs.argtypes = _GRID + [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
    ok = L.oracle_tabg_rhs(*_grid(table, 10), y.ctypes.data, d.ctypes.data, C.byref(H), kappa, C.byref(E))
    return (d, H.value, E.value) if ok else None


def integrate_general(table: dict, state_in: np.ndarray, h: float, nsteps: int, r_capture: float = -np.inf,
                      r_escape: float = np.inf, kind: int = TIMELIKE, flags: int = 0, long_double: bool = False,
                      nthreads: int = 1, snapshot_every: int = 0, snap_capacity: int | None = None, snap_mask: int = 0xFF) -> dict:
    """Fixed-step RK4 through a general ten-field tabulated metric (reading T6); trajectory records as in integrate()."""
    st = np.ascontiguousarray(state_in, dtype=np.float64)
    n = st.shape[1]
    res = {"final_state": np.full((8, n), np.nan), "status": np.full(n, -1, dtype=np.int32),
           "steps_done": np.zeros(n, dtype=np.int64), "eq_cross_r": np.full(n, np.nan), "health": np.full(n, np.nan),
           "snapshots": None, "snap_count": None}
    if snapshot_every > 0:
        if snap_capacity is None:
            snap_capacity = 1 + nsteps // snapshot_every
        res["snapshots"] = np.full((n, snap_capacity, bin(snap_mask & 0xFF).count("1")), np.nan)
        res["snap_count"] = np.zeros(n, dtype=np.int32)
    stop = _Stop(r_capture, r_escape, kind, flags)
    out = _Out(res["final_state"].ctypes.data, res["status"].ctypes.data, res["steps_done"].ctypes.data,
               res["eq_cross_r"].ctypes.data, res["health"].ctypes.data,
               res["snapshots"].ctypes.data if snapshot_every > 0 else None, snap_capacity or 0, snap_mask,
               res["snap_count"].ctypes.data if snapshot_every > 0 else None)
    L = lib()
    L.oracle_tabg_integrate.restype = C.c_int
    L.oracle_tabg_integrate.argtypes = _GRID + [C.c_void_p, C.c_int64, C.c_double, C.c_int64, C.POINTER(_Stop),
                                                C.POINTER(_Out), C.c_int, C.c_int, C.c_int64]
    rc = L.oracle_tabg_integrate(*_grid(table, 10), st.ctypes.data, n, h, nsteps, C.byref(stop), C.byref(out),
                                 int(long_double), nthreads, snapshot_every)
    if rc != 0:
        raise ValueError("oracle_tabg_integrate: invalid arguments")
    return res


class _Ctl(C.Structure):
    _fields_ = [("h0", C.c_double), ("rtol", C.c_double), ("atol", C.c_double), ("h_min", C.c_double),
                ("tau_end", C.c_double), ("snap_dtau", C.c_double)]


def integrate_adaptive(table: dict, state_in: np.ndarray, h0: float, rtol: float, atol: float, max_attempts: int,
                       r_capture: float = -np.inf, r_escape: float = np.inf, kind: int = TIMELIKE, h_min: float = 1e-12,
                       tau_end: float = np.inf, long_double: bool = False, nthreads: int = 1, snap_dtau: float = 0.0,
                       snap_capacity: int = 0, snap_mask: int = 0xFF, general: bool = False) -> dict:
    """Adaptive Dormand-Prince RK5(4) (readings A1-A3) through the five-field tabulated metric (reading T7), or with
    general=True through a ten-field table (reading T6)."""
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
    fn = L.oracle_tabg_integrate_adaptive if general else L.oracle_tab_integrate_adaptive
    fn.restype = C.c_int
    fn.argtypes = _GRID + [C.c_void_p, C.c_int64, C.POINTER(_Ctl), C.c_int64, C.POINTER(_Stop),
                           C.POINTER(_Out), C.c_void_p, C.c_int, C.c_int]
    rc = fn(*_grid(table, 10 if general else 5), st.ctypes.data, n, C.byref(ctl), max_attempts, C.byref(stop),
            C.byref(out), res["rejected"].ctypes.data, int(long_double), nthreads)
    if rc != 0:
        raise ValueError("oracle_tab_integrate_adaptive: invalid arguments")
    return res


def integrate_adaptive_general(table: dict, state_in: np.ndarray, h0: float, rtol: float, atol: float, max_attempts: int,
                               **kw) -> dict:
    """Adaptive RK5(4) through a GENERAL ten-field table (readings T6 + T7)."""
    return integrate_adaptive(table, state_in, h0, rtol, atol, max_attempts, general=True, **kw)
