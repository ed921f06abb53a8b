"""Thin Python binding of libgeo.so (include/geo.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used for device memory
and streams.  There is NO CPU fallback: if the library cannot be loaded, or there is no CUDA device,
the calls raise.  Names follow the C ABI: ``geo_create``, ``geo_integrate``, ``geo_integrate_host``,
``geo_create_tabulated``, ``geo_create_tabulated_general``, ``geo_integrate_adaptive``, ``geo_integrate_adaptive_host``, ``geo_destroy``, ``geo_horizon_radius``,
``geo_last_error``, the allocation-free ``geo_integrate_host_noalloc`` / ``geo_noalloc_last_error``; plus the development helpers of include/geo_dev.h (``geo_launch_info``, ``geo_probe_dfma``) used by bench.py.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

SCHWARZSCHILD, KERR, TABULATED, TABULATED_GENERAL, KERR_SCHILD = 0, 1, 2, 3, 4
TIMELIKE, NULL = 0, 1
OK, EINVAL, ECUDA, ENOMEM = 0, 1, 2, 3
ST_MAXSTEPS, ST_CAPTURED, ST_ESCAPED, ST_NUMERIC, ST_OUTSIDE = 0, 1, 2, 3, 4
FLAG_PLAIN_UPDATE, FLAG_STATIC_MAP, FLAG_STAGED_SNAP, FLAG_CARTESIAN_SNAP, FLAG_TAB_GATHER = 1, 2, 4, 8, 16

NOALLOC_MAX_N = 65536   # GEO_NOALLOC_MAX_N: particles per geo_integrate_host_noalloc call (size of the static scratch)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("GEO_LIB") or os.path.join(_HERE, "libgeo.so")   # GEO_LIB: load another build of the same ABI

# every symbol include/geo.h declares, then the development helpers of include/geo_dev.h
SYMBOLS = ("geo_create", "geo_create_tabulated", "geo_create_tabulated_general", "geo_integrate", "geo_integrate_host", "geo_integrate_adaptive", "geo_integrate_adaptive_host", "geo_destroy",
           "geo_horizon_radius", "geo_last_error", "geo_integrate_host_noalloc", "geo_noalloc_last_error")
DEV_SYMBOLS = ("geo_launch_info", "geo_probe_dfma")


class GeoStop(C.Structure):
    _fields_ = [("r_capture", C.c_double), ("r_escape", C.c_double), ("kind", C.c_int32), ("flags", C.c_int32)]


class GeoOut(C.Structure):
    _fields_ = [("final_state", C.c_void_p), ("status", C.c_void_p), ("steps_done", C.c_void_p),
                ("eq_cross_r", C.c_void_p), ("health", C.c_void_p), ("snapshots", C.c_void_p),
                ("snap_capacity", C.c_int64), ("snap_mask", C.c_uint32), ("snap_count", C.c_void_p),
                ("coarse_steps", C.c_void_p)]


class GeoAdaptive(C.Structure):
    _fields_ = [("h0", C.c_double), ("rtol", C.c_double), ("atol", C.c_double), ("h_min", C.c_double),
                ("tau_end", C.c_double), ("snap_dtau", C.c_double)]


class GeoTable(C.Structure):
    _fields_ = [("tab", C.c_void_p), ("n1", C.c_int64), ("n2", C.c_int64), ("x1_0", C.c_double), ("d1", C.c_double),
                ("x2_0", C.c_double), ("d2", C.c_double)]


class GeoError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libgeo error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Load libgeo.so (built in-tree by paper_1803_08320_b200/build.py).  Fails loudly if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1803_08320_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.geo_create.restype = C.c_int
        L.geo_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double]
        L.geo_create_tabulated.restype = C.c_int
        L.geo_create_tabulated.argtypes = [C.POINTER(C.c_void_p), C.POINTER(GeoTable)]
        L.geo_create_tabulated_general.restype = C.c_int
        L.geo_create_tabulated_general.argtypes = [C.POINTER(C.c_void_p), C.POINTER(GeoTable)]
        L.geo_integrate.restype = C.c_int
        L.geo_integrate.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_int64,
                                    C.POINTER(GeoStop), C.c_int64, C.POINTER(GeoOut), C.c_void_p]
        L.geo_integrate_host.restype = C.c_int
        L.geo_integrate_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_int64,
                                         C.POINTER(GeoStop), C.c_int64, C.POINTER(GeoOut)]
        L.geo_integrate_adaptive.restype = C.c_int
        L.geo_integrate_adaptive.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(GeoAdaptive), C.c_int64,
                                             C.POINTER(GeoStop), C.POINTER(GeoOut), C.c_void_p, C.c_void_p]
        L.geo_integrate_adaptive_host.restype = C.c_int
        L.geo_integrate_adaptive_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(GeoAdaptive), C.c_int64,
                                                  C.POINTER(GeoStop), C.POINTER(GeoOut), C.c_void_p]
        L.geo_destroy.restype = None
        L.geo_destroy.argtypes = [C.c_void_p]
        L.geo_horizon_radius.restype = C.c_double
        L.geo_horizon_radius.argtypes = [C.c_void_p]
        L.geo_last_error.restype = C.c_char_p
        L.geo_last_error.argtypes = [C.c_void_p]
        L.geo_integrate_host_noalloc.restype = C.c_int
        L.geo_integrate_host_noalloc.argtypes = [C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_int64, C.c_double, C.c_int64,
                                                 C.POINTER(GeoStop), C.POINTER(GeoOut), C.c_void_p]
        L.geo_noalloc_last_error.restype = C.c_char_p
        L.geo_noalloc_last_error.argtypes = []
        L.geo_launch_info.restype = C.c_int
        L.geo_launch_info.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_int64, C.POINTER(C.c_int32 * 4)]
        L.geo_probe_dfma.restype = C.c_int
        L.geo_probe_dfma.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
        _lib = L
    return _lib


def _check(ctx, rc: int):
    if rc != OK:
        raise GeoError(rc, lib().geo_last_error(ctx).decode() if ctx else "invalid arguments")


def geo_create(metric: int, M: float = 1.0, a: float = 0.0) -> C.c_void_p:
    ctx = C.c_void_p()
    rc = lib().geo_create(C.byref(ctx), metric, M, a)
    if rc != OK:
        raise GeoError(rc, "geo_create failed (invalid metric/M/a, or no CUDA device)")
    return ctx


def geo_create_tabulated(tab: np.ndarray, x1_0: float, d1: float, x2_0: float, d2: float) -> C.c_void_p:
    """Context for a tabulated 3+1 metric (include/geo.h: geo_create_tabulated).  ``tab``: host float64 [5][n2][n1] =
    alpha, beta^phi, gamma_11, gamma_22, gamma_33 at the grid nodes; it is copied to the device."""
    if not (isinstance(tab, np.ndarray) and tab.dtype == np.float64 and tab.ndim == 3 and tab.shape[0] == 5
            and tab.flags.c_contiguous):
        raise ValueError("tab must be a C-contiguous float64 numpy array of shape [5][n2][n1]")
    ctx = C.c_void_p()
    tb = GeoTable(tab.ctypes.data, tab.shape[2], tab.shape[1], x1_0, d1, x2_0, d2)
    rc = lib().geo_create_tabulated(C.byref(ctx), C.byref(tb))
    if rc != OK:
        raise GeoError(rc, "geo_create_tabulated failed (invalid table/grid, out of memory, or no CUDA device)")
    return ctx


def geo_create_tabulated_general(tab: np.ndarray, x1_0: float, d1: float, x2_0: float, d2: float) -> C.c_void_p:
    """Context for a GENERAL tabulated 3+1 metric (include/geo.h: geo_create_tabulated_general).  ``tab``: host float64
    [10][n2][n1] = alpha, beta^1, beta^2, beta^3, gamma_11, gamma_12, gamma_13, gamma_22, gamma_23, gamma_33."""
    if not (isinstance(tab, np.ndarray) and tab.dtype == np.float64 and tab.ndim == 3 and tab.shape[0] == 10
            and tab.flags.c_contiguous):
        raise ValueError("tab must be a C-contiguous float64 numpy array of shape [10][n2][n1]")
    ctx = C.c_void_p()
    tb = GeoTable(tab.ctypes.data, tab.shape[2], tab.shape[1], x1_0, d1, x2_0, d2)
    rc = lib().geo_create_tabulated_general(C.byref(ctx), C.byref(tb))
    if rc != OK:
        raise GeoError(rc, "geo_create_tabulated_general failed (invalid table/grid, out of memory, or no CUDA device)")
    return ctx


def geo_destroy(ctx) -> None:
    lib().geo_destroy(ctx)


def geo_horizon_radius(ctx) -> float:
    return lib().geo_horizon_radius(ctx)


def geo_last_error(ctx) -> str:
    return lib().geo_last_error(ctx).decode()


def geo_launch_info(ctx, n: int, flags: int = 0, snapshot_every: int = 0) -> dict:
    info = (C.c_int32 * 4)()
    _check(ctx, lib().geo_launch_info(ctx, n, flags, snapshot_every, C.byref(info)))
    return {"grid": info[0], "block": info[1], "regs": info[2], "ctas_per_sm": info[3]}


def _ncomp(mask: int) -> int:
    return bin(mask & 0xFF).count("1")


def alloc_outputs(n: int, device, nsteps: int = 0, snapshot_every: int = 0, snap_capacity: int | None = None,
                  snap_mask: int = 0xFF, want_eq_cross: bool = True, want_health: bool = True,
                  want_coarse: bool = False) -> dict:
    """Caller-owned device output tensors for geo_integrate (torch = device memory only)."""
    import torch
    out = {
        "final_state": torch.empty((8, n), dtype=torch.float64, device=device),
        "status": torch.full((n,), -1, dtype=torch.int32, device=device),
        "steps_done": torch.zeros((n,), dtype=torch.int64, device=device),
        "eq_cross_r": torch.empty((n,), dtype=torch.float64, device=device) if want_eq_cross else None,
        "health": torch.empty((n,), dtype=torch.float64, device=device) if want_health else None,
        "snapshots": None, "snap_count": None, "snap_capacity": 0, "snap_mask": snap_mask,
        "coarse_steps": torch.zeros((n,), dtype=torch.int32, device=device) if want_coarse else None,
    }
    if snapshot_every > 0:
        cap = snap_capacity if snap_capacity is not None else 1 + nsteps // snapshot_every
        out["snap_capacity"] = cap
        out["snapshots"] = torch.full((n, cap, _ncomp(snap_mask)), float("nan"), dtype=torch.float64, device=device)
        out["snap_count"] = torch.zeros((n,), dtype=torch.int32, device=device)
    return out


def _ptr(x):
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


def _out_struct(out: dict) -> GeoOut:
    return GeoOut(_ptr(out["final_state"]), _ptr(out["status"]), _ptr(out["steps_done"]),
                  _ptr(out.get("eq_cross_r")), _ptr(out.get("health")), _ptr(out.get("snapshots")),
                  int(out.get("snap_capacity") or 0), int(out.get("snap_mask", 0xFF)), _ptr(out.get("snap_count")),
                  _ptr(out.get("coarse_steps")))


_OUT_DTYPES = {"final_state": "float64", "status": "int32", "steps_done": "int64", "eq_cross_r": "float64",
               "health": "float64", "snapshots": "float64", "snap_count": "int32", "coarse_steps": "int32"}


def _check_buffers(state_in, out: dict, device: bool, rejected=None) -> int:
    """Shape / dtype / contiguity checks of the caller's buffers (the C ABI sees raw pointers only).  Returns n."""
    def props(x):
        if isinstance(x, np.ndarray):
            return (not device), str(x.dtype), x.flags.c_contiguous, tuple(x.shape), x.size
        return (x.is_cuda == device), str(x.dtype).replace("torch.", ""), x.is_contiguous(), tuple(x.shape), x.numel()
    where = "CUDA" if device else "host (numpy / CPU tensor)"
    ok, dt, cont, shape, _ = props(state_in)
    if not (ok and dt == "float64" and cont and len(shape) == 2 and shape[0] == 6):
        raise ValueError(f"state_in must be a contiguous {where} float64 array of shape [6][n]")
    n = shape[1]
    ncomp = _ncomp(int(out.get("snap_mask", 0xFF)))
    need = {"final_state": 8 * n, "status": n, "steps_done": n, "eq_cross_r": n, "health": n, "snap_count": n,
            "coarse_steps": n, "snapshots": n * int(out.get("snap_capacity") or 0) * ncomp}
    for k, want in _OUT_DTYPES.items():
        v = out.get(k)
        if v is None:
            if k in ("final_state", "status", "steps_done"):
                raise ValueError(f"out['{k}'] is required")
            continue
        ok, dt, cont, _, size = props(v)
        if not (ok and dt == want and cont and size >= need[k]):
            raise ValueError(f"out['{k}'] must be a contiguous {where} {want} array with >= {need[k]} elements")
    if rejected is not None:
        ok, dt, cont, _, size = props(rejected)
        if not (ok and dt == "int32" and cont and size >= n):
            raise ValueError(f"rejected must be a contiguous {where} int32 array with >= {n} elements")
    return n


def geo_integrate(ctx, state_in, h: float, nsteps: int, out: dict, r_capture: float = -float("inf"),
                  r_escape: float = float("inf"), kind: int = TIMELIKE, flags: int = 0,
                  snapshot_every: int = 0, stream=None) -> None:
    """Enqueue the integration of the geodesics in ``state_in`` (CUDA float64 tensor [6][n]) on
    ``stream`` (torch.cuda.Stream; default: the current stream).  Does not synchronise."""
    import torch
    n = _check_buffers(state_in, out, device=True)
    s = stream if stream is not None else torch.cuda.current_stream(state_in.device)
    stop = GeoStop(r_capture, r_escape, kind, flags)
    o = _out_struct(out)
    with torch.cuda.device(state_in.device):
        rc = lib().geo_integrate(ctx, state_in.data_ptr(), n, h, nsteps, C.byref(stop), snapshot_every,
                                 C.byref(o), C.c_void_p(s.cuda_stream))
    _check(ctx, rc)


def geo_integrate_adaptive(ctx, state_in, h0: float, rtol: float, atol: float, max_attempts: int, out: dict,
                           r_capture: float = -float("inf"), r_escape: float = float("inf"), kind: int = TIMELIKE,
                           h_min: float = 1e-12, tau_end: float = float("inf"), rejected=None, stream=None,
                           snap_dtau: float = 0.0, flags: int = 0) -> None:
    """Enqueue the adaptive RK5(4) integration (include/geo.h: geo_integrate_adaptive).  ``rejected``: optional
    CUDA int32 tensor [n].  ``snap_dtau`` > 0: dense-output records into out["snapshots"].  Does not synchronise."""
    import torch
    n = _check_buffers(state_in, out, device=True, rejected=rejected)
    s = stream if stream is not None else torch.cuda.current_stream(state_in.device)
    stop = GeoStop(r_capture, r_escape, kind, flags)
    ctl = GeoAdaptive(h0, rtol, atol, h_min, tau_end, snap_dtau)
    o = _out_struct(out)
    L = lib()
    with torch.cuda.device(state_in.device):
        rc = L.geo_integrate_adaptive(ctx, state_in.data_ptr(), n, C.byref(ctl), max_attempts, C.byref(stop),
                                      C.byref(o), _ptr(rejected), C.c_void_p(s.cuda_stream))
    _check(ctx, rc)


def geo_integrate_adaptive_host(ctx, state_in, h0: float, rtol: float, atol: float, max_attempts: int, out: dict,
                                r_capture: float = -float("inf"), r_escape: float = float("inf"), kind: int = TIMELIKE,
                                h_min: float = 1e-12, tau_end: float = float("inf"), rejected=None,
                                snap_dtau: float = 0.0, flags: int = 0) -> None:
    """The adaptive RK5(4) integration on HOST buffers (numpy arrays or pinned CPU tensors); synchronous."""
    n = _check_buffers(state_in, out, device=False, rejected=rejected)
    stop = GeoStop(r_capture, r_escape, kind, flags)
    ctl = GeoAdaptive(h0, rtol, atol, h_min, tau_end, snap_dtau)
    o = _out_struct(out)
    L = lib()
    _check(ctx, L.geo_integrate_adaptive_host(ctx, _ptr(state_in), n, C.byref(ctl), max_attempts, C.byref(stop),
                                              C.byref(o), _ptr(rejected)))


def geo_integrate_host(ctx, state_in: np.ndarray, h: float, nsteps: int, out: dict,
                       r_capture: float = -float("inf"), r_escape: float = float("inf"),
                       kind: int = TIMELIKE, flags: int = 0, snapshot_every: int = 0) -> None:
    """Same operation on HOST buffers (numpy arrays or pinned CPU tensors); synchronous."""
    n = _check_buffers(state_in, out, device=False)
    stop = GeoStop(r_capture, r_escape, kind, flags)
    o = _out_struct(out)
    rc = lib().geo_integrate_host(ctx, _ptr(state_in), n, h, nsteps, C.byref(stop), snapshot_every, C.byref(o))
    _check(ctx, rc)


def geo_noalloc_last_error() -> str:
    return lib().geo_noalloc_last_error().decode()


def geo_integrate_host_noalloc(metric: int, M: float, a: float, state_in: np.ndarray, h: float, nsteps: int, out: dict,
                               r_capture: float = -float("inf"), r_escape: float = float("inf"),
                               kind: int = TIMELIKE, flags: int = 0, stream=None) -> None:
    """geo_integrate_host without a ctx and without any device allocation (static device scratch inside the library,
    at most NOALLOC_MAX_N particles per call, no trajectory records); synchronous.  stream: a torch.cuda.Stream or None."""
    n = _check_buffers(state_in, out, device=False)
    stop = GeoStop(r_capture, r_escape, kind, flags)
    o = _out_struct(out)
    rc = lib().geo_integrate_host_noalloc(metric, M, a, _ptr(state_in), n, h, nsteps, C.byref(stop), C.byref(o),
                                          C.c_void_p(stream.cuda_stream) if stream is not None else None)
    if rc != OK:
        raise GeoError(rc, geo_noalloc_last_error())


def alloc_outputs_host(n: int, nsteps: int = 0, snapshot_every: int = 0, snap_capacity: int | None = None,
                       snap_mask: int = 0xFF, want_eq_cross: bool = True, want_health: bool = True,
                       pinned: bool = False, want_coarse: bool = False) -> dict:
    """Host output buffers for geo_integrate_host (numpy, or pinned torch CPU tensors)."""
    if pinned:
        import torch

        def mk(shape, dt, fill=None):
            t = torch.empty(shape, dtype=dt, pin_memory=True)
            if fill is not None:
                t.fill_(fill)
            return t
        f64, i32, i64 = torch.float64, torch.int32, torch.int64
    else:
        def mk(shape, dt, fill=None):
            a = np.empty(shape, dtype=dt)
            if fill is not None:
                a.fill(fill)
            return a
        f64, i32, i64 = np.float64, np.int32, np.int64
    out = {
        "final_state": mk((8, n), f64), "status": mk((n,), i32, -1), "steps_done": mk((n,), i64, 0),
        "eq_cross_r": mk((n,), f64) if want_eq_cross else None,
        "health": mk((n,), f64) if want_health else None,
        "snapshots": None, "snap_count": None, "snap_capacity": 0, "snap_mask": snap_mask,
        "coarse_steps": mk((n,), i32, 0) if want_coarse else None,
    }
    if snapshot_every > 0:
        cap = snap_capacity if snap_capacity is not None else 1 + nsteps // snapshot_every
        out["snap_capacity"] = cap
        out["snapshots"] = mk((n, cap, _ncomp(snap_mask)), f64, float("nan"))
        out["snap_count"] = mk((n,), i32, 0)
    return out


def geo_probe_dfma(ctx, iters: int, sink, stream=None) -> float:
    """Enqueue the register-only DFMA throughput probe; returns the number of FMAs it executes."""
    import torch
    s = stream if stream is not None else torch.cuda.current_stream(sink.device)
    n_fma = C.c_double()
    _check(ctx, lib().geo_probe_dfma(ctx, iters, sink.data_ptr(), C.byref(n_fma), C.c_void_p(s.cuda_stream)))
    return n_fma.value


def to_numpy(out: dict) -> dict:
    """Copy a dict of device outputs to host numpy arrays (after the caller synchronised)."""
    res = {}
    for k, v in out.items():
        if v is None or isinstance(v, (int, float)):
            res[k] = v
        elif isinstance(v, np.ndarray):
            res[k] = v
        else:
            res[k] = v.cpu().numpy()
    return res
