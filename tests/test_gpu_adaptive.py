"""GPU parity of the adaptive RK5(4) path (include/geo.h: geo_integrate_adaptive) with the
oracle's, element by element on the same seeded inputs.

Both sides take every accept/reject decision in FP64, but on error estimates whose rounding differs (the
estimate is a cancelling sum of stage derivatives: its relative noise is ~1e-16 |k| h / (rtol |y|)), so a
decision can flip for a ray whose err lands within that noise of 1.  What is unique is compared strictly
(termination class; state at the common final time within the integrator's tolerance), what is not (the
number of accepted / rejected steps) is checked to agree for nearly all particles and to be valid for all.
"""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import parity  # noqa: E402

from paper_1803_08320_b200 import workloads as W  # noqa: E402

pytestmark = pytest.mark.gpu
NCPU = max(1, (os.cpu_count() or 1))


def run_gpu_adaptive(G, metric, a, st, h0, rtol, atol, max_attempts, M=1.0, **kw):
    import torch
    dev = torch.device("cuda:0")
    ctx = G.geo_create(metric, M, a)
    try:
        n = st.shape[1]
        d_in = torch.from_numpy(np.ascontiguousarray(st)).to(dev)
        out = G.alloc_outputs(n, dev)
        rej = torch.full((n,), -1, dtype=torch.int32, device=dev)
        G.geo_integrate_adaptive(ctx, d_in, h0, rtol, atol, max_attempts, out, rejected=rej, **kw)
        torch.cuda.synchronize()
        g = G.to_numpy(out)
        g["rejected"] = rej.cpu().numpy()
        return g
    finally:
        G.geo_destroy(ctx)


def test_fixed_step_mode_is_the_plain_fifth_order_method(G, oracle):
    """rtol = inf: no decisions at all, so parity must be as tight as for RK4 (1e-9), steps identical."""
    a = 0.9
    st = W.kerr_bound(1000, a, W.SEED_BASE + 2)
    o = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.05, np.inf, 1.0, 4000, nthreads=NCPU)
    g = run_gpu_adaptive(G, G.KERR, a, st, 0.05, float("inf"), 1.0, 4000)
    c = parity.compare(g, o)
    assert c["same_class"].all() and (g["steps_done"] == 4000).all() and (g["rejected"] == 0).all()
    assert c["err"].max() <= 1e-9, c["err"].max()


@pytest.mark.parametrize("metric_a", [0.0, 0.9])
def test_adaptive_bound_orbits_to_a_final_time(G, oracle, metric_a):
    a = metric_a
    if a:
        st, metric, ometric = W.kerr_bound(3000, a, W.SEED_BASE + 2), G.KERR, oracle.KERR
    else:
        st, metric, ometric = W.circular_schwarzschild(3000), G.SCHWARZSCHILD, oracle.SCHWARZSCHILD
        st[3] = 0.02                                   # a radial kick: eccentric orbits
    kw = dict(tau_end=500.0)
    o = oracle.integrate_adaptive(ometric, 1.0, a, st, 0.01, 1e-12, 1e-12, 200000, nthreads=NCPU, **kw)
    g = run_gpu_adaptive(G, metric, a, st, 0.01, 1e-12, 1e-12, 200000, **kw)
    assert np.array_equal(g["status"], o["status"]) and (g["status"] == G.ST_MAXSTEPS).all()
    e = parity.rel_err(g["final_state"], o["final_state"]).max(axis=0)
    assert e.max() <= 1e-9, e.max()
    same = (g["steps_done"] == o["steps_done"]) & (g["rejected"] == o["rejected"])
    assert same.mean() > 0.98, same.mean()
    assert (np.abs(g["steps_done"] - o["steps_done"]) <= 3).all()
    assert g["health"].max() < 1e-9


def test_adaptive_camera_rays_classes_and_finals(G, oracle):
    """Config-3-shaped rays (a = 0.998, i = 60 deg) to tau_end = 1015 or capture: class identical, state at the
    final time within 1e-8 on certified rays (double vs long double oracle), ~100x fewer steps than RK4."""
    a = 0.998
    full = W.camera_rays(1024, a, 60.0)
    ii = np.arange(1024 * 1024).reshape(1024, 1024)[7::31, 5::31].ravel()
    st = np.ascontiguousarray(full[:, ii])
    rc = W.horizon_radius(1.0, a) + 0.01
    kw = dict(r_capture=rc, r_escape=1100.0, tau_end=1015.0)
    o = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.02, 1e-11, 1e-11, 100000, kind=oracle.NULL, nthreads=NCPU, **kw)
    o_ld = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.02, 1e-11, 1e-11, 100000, kind=oracle.NULL, nthreads=NCPU,
                                     long_double=True, **kw)
    g = run_gpu_adaptive(G, G.KERR, a, st, 0.02, 1e-11, 1e-11, 100000, kind=G.NULL, **kw)
    assert set(np.unique(o["status"])) == {oracle.ST_MAXSTEPS, oracle.ST_CAPTURED}
    # a captured ray's record is its last accepted state, which depends on the step sequence: class only
    cert = (o["status"] == o_ld["status"]) & ((o["status"] == oracle.ST_CAPTURED) |
                                              (parity.rel_err(o["final_state"], o_ld["final_state"]).max(axis=0) <= 1e-9))
    assert cert.mean() > 0.97
    assert (g["status"] == o["status"])[cert].all() and (g["status"] != o["status"]).sum() <= 1
    alive = cert & (o["status"] == oracle.ST_MAXSTEPS)
    e = parity.rel_err(g["final_state"][:, alive], o["final_state"][:, alive]).max(axis=0)
    assert e.max() <= 1e-8, e.max()
    assert g["steps_done"][alive].max() < 3000 and g["health"][alive].max() < 1e-8
    assert np.array_equal(np.isnan(g["eq_cross_r"][alive]), np.isnan(o["eq_cross_r"][alive]))


def test_adaptive_argument_errors(G):
    import torch
    dev = torch.device("cuda:0")
    ctx = G.geo_create(G.KERR, 1.0, 0.5)
    st = torch.from_numpy(W.kerr_bound(8, 0.5, 1)).to(dev)
    out = G.alloc_outputs(8, dev)
    for bad in (dict(h0=0.0), dict(h0=-0.1), dict(rtol=0.0, atol=0.0), dict(rtol=-1.0), dict(tau_end=0.0), dict(max_attempts=-1)):
        args = dict(h0=0.01, rtol=1e-9, atol=1e-9, max_attempts=10)
        kw = {}
        for k, v in bad.items():
            (args if k in args else kw)[k] = v
        with pytest.raises(G.GeoError) as ei:
            G.geo_integrate_adaptive(ctx, st, args["h0"], args["rtol"], args["atol"], args["max_attempts"], out, **kw)
        assert ei.value.code == G.EINVAL
    G.geo_destroy(ctx)


def test_adaptive_whole_image_classes_match_the_analytic_criterion(G):
    """All 1024^2 rays of config 3 with the adaptive stepper (rtol = atol = 1e-9) against the closed-form
    capture/escape criterion -- no oracle involved.  Unlike fixed-step RK4 (reading B7) the step control also
    resolves the passages next to the polar axis."""
    from test_gpu_fullsize import _escapes_analytic
    a, N = 0.998, 1024
    st, (al, be, Lz, Q) = W.camera_rays(N, a, 60.0, return_constants=True)
    rp = W.horizon_radius(1.0, a)
    g = run_gpu_adaptive(G, G.KERR, a, st, 0.02, 1e-9, 1e-9, 200000, kind=G.NULL, r_capture=rp + 0.01, r_escape=1100.0)
    esc = _escapes_analytic(a, Lz, Q, rp, 1000.0)
    wrong = (g["status"] == G.ST_ESCAPED) != esc
    print("adaptive: mismatches", int(wrong.sum()), "statuses", np.bincount(g["status"], minlength=4).tolist(),
          "mean accepted steps", float(g["steps_done"].mean()), "mean rejected", float(g["rejected"].mean()))
    assert np.isin(g["status"], (G.ST_CAPTURED, G.ST_ESCAPED)).all()
    assert wrong.sum() <= 4                       # measured: 0 of 1 048 576


def test_adaptive_host_entry_point_equals_the_device_one(G):
    """geo_integrate_adaptive_host (H2D, launch, D2H inside the C ABI) returns bit for bit what the device entry point does."""
    a = 0.998
    full = W.camera_rays(256, a, 60.0)
    ii = np.arange(256 * 256).reshape(256, 256)[3::5, 1::5].ravel()
    st = np.ascontiguousarray(full[:, ii])
    rp = W.horizon_radius(1.0, a)
    g = run_gpu_adaptive(G, G.KERR, a, st, 0.02, 1e-9, 1e-9, 200000, kind=G.NULL, r_capture=rp + 0.01, r_escape=1100.0)
    ctx = G.geo_create(G.KERR, 1.0, a)
    out = G.alloc_outputs_host(st.shape[1])
    rej = np.zeros(st.shape[1], dtype=np.int32)
    G.geo_integrate_adaptive_host(ctx, st, 0.02, 1e-9, 1e-9, 200000, out, kind=G.NULL, r_capture=rp + 0.01, r_escape=1100.0,
                                  rejected=rej)
    G.geo_destroy(ctx)
    for k in ("final_state", "status", "steps_done", "eq_cross_r", "health"):
        assert np.array_equal(np.asarray(out[k]), g[k], equal_nan=True), k
    assert np.array_equal(rej, g["rejected"])



def test_undefined_error_estimate_ends_with_numeric_not_after_max_attempts(G, oracle):
    """Reading A2 (round 2, advisor finding): an attempt whose error estimate is NaN (atol = 0 on the exactly-zero phi
    of a radial infall) is rejected with factor 0.2; the particle ends with NUMERIC once the step is below h_min, or has
    shrunk to exactly zero with h_min = 0 -- after the same number of rejections as in the oracle, not after
    max_attempts = 10^6 futile retries."""
    st = np.zeros((6, 40))
    st[0] = np.linspace(6.0, 30.0, 40)
    st[1] = np.pi / 2
    st[3] = -0.1
    for h_min in (1e-12, 0.0):
        kw = dict(h_min=h_min)
        o = oracle.integrate_adaptive(oracle.SCHWARZSCHILD, 1.0, 0.0, st, 0.1, 1e-9, 0.0, 10**6, **kw)
        g = run_gpu_adaptive(G, G.SCHWARZSCHILD, 0.0, st, 0.1, 1e-9, 0.0, 10**6, **kw)
        assert (o["status"] == oracle.ST_NUMERIC).all() and (g["status"] == G.ST_NUMERIC).all()
        assert np.array_equal(g["rejected"], o["rejected"]) and (g["steps_done"] == 0).all()
        assert np.array_equal(g["final_state"][1:4], st[0:3])


# ---- reading A3: dense output (records at fixed tau from the pair's continuous extension) ---------------------------
def run_gpu_dense(G, metric, a, st, h0, rtol, atol, max_attempts, snap_dtau, cap, mask=0xFF, flags=0, host=False, **kw):
    import torch
    ctx = G.geo_create(metric, 1.0, a)
    try:
        n = st.shape[1]
        if host:
            out = G.alloc_outputs_host(n, 0, 1, cap, mask)
            rej = np.full(n, -1, dtype=np.int32)
            G.geo_integrate_adaptive_host(ctx, np.ascontiguousarray(st), h0, rtol, atol, max_attempts, out, rejected=rej,
                                          snap_dtau=snap_dtau, flags=flags, **kw)
            g = G.to_numpy(out)
            g["rejected"] = rej
            return g
        dev = torch.device("cuda:0")
        out = G.alloc_outputs(n, dev, 0, 1, cap, mask)
        rej = torch.full((n,), -1, dtype=torch.int32, device=dev)
        G.geo_integrate_adaptive(ctx, torch.from_numpy(np.ascontiguousarray(st)).to(dev), h0, rtol, atol, max_attempts, out,
                                 rejected=rej, snap_dtau=snap_dtau, flags=flags, **kw)
        torch.cuda.synchronize()
        g = G.to_numpy(out)
        g["rejected"] = rej.cpu().numpy()
        return g
    finally:
        G.geo_destroy(ctx)


@pytest.mark.parametrize("mask,flags", [(0xFF, 0), (0x0F, 8), (0x07, 0)])
def test_dense_output_fixed_step_mode_vs_oracle(G, oracle, mask, flags):
    """rtol = inf: identical step sequences on both sides, so every record -- interpolated inside the steps, the record
    times are not multiples of h -- must agree like the states themselves (1e-9; measured ~1e-13), also in the paper's
    (t, x, y, z) format and with an odd component count; capacity overflow drops but counts (S3)."""
    a = 0.9
    st = W.kerr_bound(1500, a, W.SEED_BASE + 2)
    kw = dict(tau_end=60.0)
    for cap in (100, 7):
        o = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.05, np.inf, 1.0, 10**6, snap_dtau=0.7, snap_capacity=cap,
                                      snap_mask=mask, flags=flags, nthreads=NCPU, **kw)
        g = run_gpu_dense(G, G.KERR, a, st, 0.05, float("inf"), 1.0, 10**6, 0.7, cap, mask, flags, **kw)
        c = parity.compare(g, o)
        assert c["same_class"].all() and c["err"].max() <= 1e-9
        assert np.array_equal(g["snap_count"], o["snap_count"]) and (g["snap_count"] == 1 + int(60.0 / 0.7)).all()
        e = parity.snapshot_err(g, o)
        assert e.max() <= 1e-9, e.max()
        valid = np.arange(cap)[None, :] < np.minimum(g["snap_count"], cap)[:, None]
        assert np.isnan(g["snapshots"][~valid]).all() and np.isfinite(g["snapshots"][valid]).all()


def test_dense_output_adaptive_bound_orbits_and_host_entry(G, oracle):
    """Step control on (rtol = atol = 1e-11): the two sides may choose different step sequences, the records approximate
    the same solution to the integrator's tolerance: 1e-8.  The host entry point (chunk pipeline) returns the device
    path's bits."""
    a = 0.9
    st = W.kerr_bound(3001, a, W.SEED_BASE + 2)
    args = (0.05, 1e-11, 1e-11, 10**6)
    kw = dict(tau_end=200.0)
    o = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, *args, snap_dtau=2.5, snap_capacity=81, nthreads=NCPU, **kw)
    g = run_gpu_dense(G, G.KERR, a, st, *args, 2.5, 81, **kw)
    assert (g["status"] == G.ST_MAXSTEPS).all() and np.array_equal(g["snap_count"], o["snap_count"]) and (g["snap_count"] == 81).all()
    # reading P3: every orbit the oracle itself determines to 1e-9 (long double run, 1-ulp-nudged run) is within 1e-8 --
    # final state and all 81 records; the few low-|L_z| orbits that are not are counted and printed
    def certify(jj):
        sub = np.ascontiguousarray(st[:, jj])
        okw = dict(snap_dtau=2.5, snap_capacity=81, nthreads=NCPU, **kw)
        runs = [oracle.integrate_adaptive(oracle.KERR, 1.0, a, sub, *args, long_double=True, **okw),
                oracle.integrate_adaptive(oracle.KERR, 1.0, a, parity.ulp_nudged(sub), *args, **okw)]
        for r_ in runs:                       # same conventions as for the GPU comparison
            r_["eq_cross_r"] = None
            r_["steps_done"] = o["steps_done"][jj]
        return runs
    og = dict(o)
    og["steps_done"] = g["steps_done"]        # step counts may differ (controller noise): the class here is the status
    # eq_cross_r is a LINEAR interpolation between the two accepted states that bracket the crossing: an O(h^2) quantity
    # that depends on where the accepted states lie.  Even with equal accept/reject COUNTS the step SIZES differ by the
    # controller's ~1e-8 relative noise, so it is compared at 1e-6 and only where the counts agree.
    same_seq = (g["steps_done"] == o["steps_done"]) & (g["rejected"] == o["rejected"])
    assert parity.rel_err(g["eq_cross_r"], o["eq_cross_r"])[same_seq].max() <= 1e-6 and same_seq.mean() > 0.9
    og["eq_cross_r"] = None
    rep = parity.p3_report(g, og, certify, 1e-8, labels=st[[0, 1, 3, 4, 5]], max_fail_frac=0.005, what="adaptive dense bound orbits",
                           extra_err=parity.snapshot_err(g, o),
                           extra_err_fn=lambda x, y: np.where(x["status"] == y["status"], parity.snapshot_err(x, y), np.inf))
    print(rep)
    gh = run_gpu_dense(G, G.KERR, a, st, *args, 2.5, 81, host=True, **kw)
    for k in ("final_state", "status", "steps_done", "snapshots", "snap_count", "rejected", "eq_cross_r"):
        assert np.array_equal(g[k], gh[k], equal_nan=True), k


def test_dense_output_camera_rays_records_stop_with_the_ray(G, oracle):
    """Null rays with capture / escape: records exist up to the last accepted state of each ray and no further; rays whose
    accept/reject sequence is the oracle's have the oracle's record count and records within 1e-8 (t, r: the same
    remark as for the final state -- the step-size noise moves the termination point, not the records before it)."""
    a = 0.998
    full = W.camera_rays(1024, a, 60.0)
    st = np.ascontiguousarray(full[:, np.arange(1024 * 1024).reshape(1024, 1024)[200:824:13, 200:824:13].ravel()])
    kw = dict(r_capture=W.horizon_radius(1.0, a) + 0.01, r_escape=1100.0)
    o = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.02, 1e-10, 1e-10, 200000, kind=oracle.NULL, snap_dtau=20.0,
                                  snap_capacity=120, snap_mask=0x0F, nthreads=NCPU, **kw)
    g = run_gpu_dense(G, G.KERR, a, st, 0.02, 1e-10, 1e-10, 200000, 20.0, 120, 0x0F, kind=G.NULL, **kw)
    assert np.array_equal(g["status"], o["status"])
    same = (g["steps_done"] == o["steps_done"]) & (g["rejected"] == o["rejected"])
    assert same.mean() > 0.95
    assert np.array_equal(g["snap_count"][same], o["snap_count"][same])
    assert (np.abs(g["snap_count"].astype(int) - o["snap_count"]) <= 1).all()
    e = parity.snapshot_err(parity.take(g, np.flatnonzero(same)), parity.take(o, np.flatnonzero(same)))
    print("dense camera rays: same sequence", same.mean(), "max record err", e.max())
    assert e.max() <= 1e-8
    cnt = g["snap_count"]
    for i in range(0, st.shape[1], 97):
        assert np.isfinite(g["snapshots"][i, : cnt[i]]).all() and np.isnan(g["snapshots"][i, cnt[i]:]).all()
