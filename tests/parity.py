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


def take(res: dict, ii) -> dict:
    """Entries ii of every per-particle array of an oracle / GPU result dict (particle axis: last for final_state,
    first otherwise)."""
    out = {}
    for k, v in res.items():
        if isinstance(v, np.ndarray):
            out[k] = v[:, ii] if k == "final_state" else v[ii]
        else:
            out[k] = v
    return out


def snapshot_err(g: dict, o: dict) -> np.ndarray:
    """Per-particle worst P2 error over the records both sides produced; inf where the record counts differ."""
    cap = o["snapshots"].shape[1]
    valid = np.arange(cap)[None, :] < np.minimum(o["snap_count"], cap)[:, None]
    e = np.where(valid[:, :, None], rel_err(g["snapshots"], o["snapshots"]), 0.0).max(axis=(1, 2))
    return np.where(g["snap_count"] == o["snap_count"], e, np.inf)


def p3_report(g: dict, o: dict, run_certify, tol: float, labels=None, max_fail_frac: float = 0.03,
              what: str = "", extra_err=None, extra_err_fn=None) -> dict:
    """DESIGN.md reading P3 on a set of particles (null rays at 1e-8, timelike at 1e-9), evaluated lazily.

    The rule: every CERTIFIED particle must have the GPU's class (status AND steps_done) and be within tol.  A particle
    is certified iff the ORACLE ALONE determines its result to tol/10: every certification run -- the long double build,
    and (round 2) the double build started from initial data moved by one ulp -- has the oracle's class and agrees with
    it within tol/10.  Equivalently: every particle that FAILS (class or tolerance) must be uncertified, so the
    certification runs are only needed on the failing ones.  ``run_certify(ii)`` returns the list of certification
    results for the particles ii (it uses the oracle only, so the rule is fixed before any GPU result exists;
    evaluating it where it matters does not change it).  ``extra_err`` / ``extra_err_fn(o_sub, o_cert)``: additional
    per-particle error (e.g. over the trajectory records) for the GPU comparison / for the certification.
    Returns counts; raises on a violation.  ``labels``: [k][n] per-particle constants printed for uncertified ones."""
    c = compare(g, o)
    if extra_err is not None:
        c["err"] = np.maximum(c["err"], extra_err)
    n = len(c["err"])
    fail = ~c["same_class"] | ~(c["err"] <= tol)
    ii = np.flatnonzero(fail)
    assert len(ii) <= max_fail_frac * n, f"{what}: {len(ii)} of {n} fail class/tolerance -- too many to be the uncertified band"
    n_cert_fail = 0
    if len(ii):
        o_sub = take(o, ii)
        runs = run_certify(ii)
        runs = runs if isinstance(runs, (list, tuple)) else [runs]
        cert = np.ones(len(ii), dtype=bool)
        p3_only = None
        for o_c in runs:
            cc = compare(o_sub, o_c)
            e = cc["err"] if extra_err_fn is None else np.maximum(cc["err"], extra_err_fn(o_sub, o_c))
            cert &= cc["same_class"] & (e <= tol / 10.0)
            if p3_only is None:
                p3_only = cert.copy()          # first run = long double: the round-1 form of the rule
        n_cert_fail = int(cert.sum())
        print(f"{what}: {len(ii)} of {n} outside class/tolerance, all must be uncertified; certified among them: {n_cert_fail} "
              f"(by the long double run alone: {int(p3_only.sum())})")
        for k, i in enumerate(ii[:24]):
            lab = "" if labels is None else " labels (" + ", ".join(f"{labels[q][i]:.6g}" for q in range(labels.shape[0])) + ")"
            print(f"   particle {i}: gpu class ({g['status'][i]}, {g['steps_done'][i]}) oracle ({o['status'][i]}, {o['steps_done'][i]}) "
                  f"err {c['err'][i]:.3e} certified {bool(cert[k])}{lab}")
        assert n_cert_fail == 0, f"{what}: {n_cert_fail} CERTIFIED particles differ from the oracle (class or > {tol})"
    return {"n": n, "class_mismatch": int((~c["same_class"]).sum()), "fail": int(len(ii)),
            "max_err_passing": float(c["err"][~fail].max()) if (~fail).any() else 0.0}


def ulp_nudged(st: np.ndarray, row: int = 3) -> np.ndarray:
    """state_in with one component (default u_r) moved to the next double: the certification perturbation of P3."""
    out = np.array(st, dtype=np.float64, copy=True)
    out[row] = np.nextafter(out[row], np.inf)
    return out


null_parity_report = p3_report
