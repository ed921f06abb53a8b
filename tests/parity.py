"""Element-by-element comparison of a CUDA-path result with the oracle's (test helper).

Tolerance form (reading P2): |x_gpu - x_or| <= tol * max(|x_or|, 1) per component, M = 1
units; NaN == NaN for eq_cross_r; status and steps_done must be EQUAL for a particle to count as
class-identical.  Holds no arithmetic of the method.
"""
from __future__ import annotations

import numpy as np


def rel_err(x_gpu: np.ndarray, x_or: np.ndarray) -> np.ndarray:
    """P2 error measure; NaN on both sides counts as 0, NaN on one side as inf."""
    x_gpu = np.asarray(x_gpu, dtype=np.float64)
    x_or = np.asarray(x_or, dtype=np.float64)
    with np.errstate(invalid="ignore"):
        e = np.abs(x_gpu - x_or) / np.maximum(np.abs(x_or), 1.0)
    both_nan = np.isnan(x_gpu) & np.isnan(x_or)
    e = np.where(both_nan, 0.0, e)
    return np.where(np.isnan(e), np.inf, e)


def compare(gpu: dict, ora: dict) -> dict:
    """Per-particle class identity and worst P2 error over final_state (+ eq_cross_r)."""
    same_class = (gpu["status"] == ora["status"]) & (gpu["steps_done"] == ora["steps_done"])
    err = rel_err(gpu["final_state"], ora["final_state"]).max(axis=0)
    if gpu.get("eq_cross_r") is not None and ora.get("eq_cross_r") is not None:
        err = np.maximum(err, rel_err(gpu["eq_cross_r"], ora["eq_cross_r"]))
    return {"same_class": same_class, "err": err}


def certified(ora_d: dict, ora_ld: dict, tol: float) -> np.ndarray:
    """DESIGN.md reading P3: a particle is certified iff the oracle's double and long double runs have
    the same class and agree within tol/10.  Uses only the oracle."""
    c = compare(ora_d, ora_ld)
    return c["same_class"] & (c["err"] <= tol / 10.0)
