"""GPU parity tests of SURVEY 8(f).3: RK4 geodesics through a TABULATED 3+1 metric (geo_create_tabulated +
geo_integrate, include/geo.h) against the tabulated-metric oracle (oracle/geo_tab_oracle.cpp), element by element on
the same seeded inputs and the same table.  Tolerances as for the analytic metrics: 1e-9 (timelike), null rays class
identical on >= 99.99 % and 1e-8 on the certified ones (P2, P3).  Plus checks of the CUDA path against
the mathematics alone (straight lines in flat space; convergence to the analytic-metric kernel)."""
import math
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import parity  # noqa: E402

from paper_1803_08320_b200 import workloads as W  # noqa: E402

pytestmark = pytest.mark.gpu
NCPU = max(1, (os.cpu_count() or 1))


def run_gpu_tab(G, tb, st, h, nsteps, host=False, flags=0, **stop):
    import torch
    ctx = G.geo_create_tabulated(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    try:
        n = st.shape[1]
        if host:
            out = G.alloc_outputs_host(n)
            G.geo_integrate_host(ctx, np.ascontiguousarray(st), h, nsteps, out, flags=flags, **stop)
            return G.to_numpy(out)
        dev = torch.device("cuda:0")
        d_in = torch.from_numpy(np.ascontiguousarray(st)).to(dev)
        out = G.alloc_outputs(n, dev)
        G.geo_integrate(ctx, d_in, h, nsteps, out, flags=flags, **stop)
        torch.cuda.synchronize()
        return G.to_numpy(out)
    finally:
        G.geo_destroy(ctx)


def assert_parity(g, o, tol):
    c = parity.compare(g, o)
    assert c["same_class"].all(), np.flatnonzero(~c["same_class"])[:10]
    assert c["err"].max() <= tol, (c["err"].max(), int(c["err"].argmax()))
    assert (parity.rel_err(g["health"], o["health"]) <= 1e-6).all() or np.nanmax(np.abs(g["health"] - o["health"])) < 1e-9


@pytest.mark.parametrize("host,flags", [(False, 0), (True, 0), (False, 1), (False, 16), (False, 17)])   # 1 = plain update, 16 = GEO_FLAG_TAB_GATHER
def test_tabulated_kerr_bound_orbits(G, tab_oracle, host, flags):
    """Config-2-like batch (Kerr a = 0.9 bound orbits, ragged count) on a 1025 x 257 Boyer-Lindquist table."""
    a = 0.9
    tb = W.kerr_metric_table(1.0, a, 1025, 257, 1.8, 40.0, 0.2, math.pi - 0.2)
    st = W.kerr_bound(3001, a, W.SEED_BASE + 2)
    o = tab_oracle.integrate(tb, st, 0.01, 3000, flags=flags & 1, nthreads=NCPU)
    g = run_gpu_tab(G, tb, st, 0.01, 3000, host=host, flags=flags)
    assert_parity(g, o, 1e-9)
    # orbits whose polar motion leaves the table's theta range end with OUTSIDE (on both sides, same step)
    assert np.isin(g["status"], (G.ST_MAXSTEPS, G.ST_OUTSIDE)).all() and (g["status"] == G.ST_MAXSTEPS).mean() > 0.9
    assert np.array_equal(g["final_state"][7], st[5])                 # p_phi constant, exactly
    assert np.nanmax(g["health"]) < 1e-6


def test_tabulated_kerr_long_run(G, tab_oracle):
    """Rounding amplification over 10^5 steps on a small batch."""
    a = 0.5
    tb = W.kerr_metric_table(1.0, a, 513, 129, 2.5, 40.0, 0.15, math.pi - 0.15)
    st = W.kerr_bound(64, a, W.SEED_BASE + 4)
    o = tab_oracle.integrate(tb, st, 0.01, 100000, nthreads=NCPU)
    g = run_gpu_tab(G, tb, st, 0.01, 100000)
    assert_parity(g, o, 1e-9)


def test_tabulated_camera_rays_log_radial(G, tab_oracle):
    """Null rays of a config-3-like camera (a = 0.998, observer at r = 50) on a log-radial table: capture, escape,
    equatorial-crossing event; class rule of reading P3 with the oracle's long double run."""
    a = 0.998
    rp = W.horizon_radius(1.0, a)
    tb = W.kerr_metric_table(1.0, a, 769, 257, math.log(0.005), math.log(60.0), 0.0, math.pi, radial="log", ghost=3)
    full = W.camera_rays(128, a, 60.0, r_obs=50.0)
    ii = np.arange(128 * 128).reshape(128, 128)[1::3, 2::3].ravel()
    s = W.to_log_radial(np.ascontiguousarray(full[:, ii]), rp)
    kw = dict(r_capture=math.log(0.01), r_escape=math.log(55.0 - rp))
    o = tab_oracle.integrate(tb, s, 0.02, 20000, kind=tab_oracle.NULL, nthreads=NCPU, **kw)
    o_ld = tab_oracle.integrate(tb, s, 0.02, 20000, kind=tab_oracle.NULL, nthreads=NCPU, long_double=True, **kw)
    g = run_gpu_tab(G, tb, s, 0.02, 20000, kind=G.NULL, **kw)
    g2 = run_gpu_tab(G, tb, s, 0.02, 20000, kind=G.NULL, flags=G.FLAG_TAB_GATHER, **kw)
    for k in ("final_state", "status", "steps_done", "eq_cross_r"):      # the stencil cache changes where the nodes are
        assert np.array_equal(g[k], g2[k], equal_nan=True), k             # read from, not one bit of the result
    cert = parity.certified(o, o_ld, 1e-8)
    c = parity.compare(g, o)
    n = s.shape[1]
    assert (~c["same_class"]).sum() <= max(1, int(1e-4 * n)), int((~c["same_class"]).sum())
    assert c["same_class"][cert].all()
    assert c["err"][cert].max() <= 1e-8, c["err"][cert].max()
    assert cert.mean() > 0.95, cert.mean()
    assert set(np.unique(g["status"])) == {G.ST_CAPTURED, G.ST_ESCAPED}


def test_tabulated_stop_rules_and_domain_exit(G, tab_oracle):
    """B1 / T4 on y0 (captured, non-finite, outside the table), nsteps = 0, and a particle that runs off the table."""
    a = 0.998
    tb = W.kerr_metric_table(1.0, a, 769, 257, math.log(0.005), math.log(60.0), 0.0, math.pi, radial="log", ghost=3)
    y0 = np.array([[1.0, -9.0, 1.0, 1.0, 1.0], [1.5, 1.5, 1.5, 1.5, -0.5], [0.0] * 5, [0.0] * 5, [0.0] * 5, [2.0] * 5])
    y0[1, 2] = float("nan")
    y0[0, 3] = 4.5
    for nsteps in (0, 50):
        o = tab_oracle.integrate(tb, y0, 0.02, nsteps, r_capture=-6.0, r_escape=9.0)
        g = run_gpu_tab(G, tb, y0, 0.02, nsteps, r_capture=-6.0, r_escape=9.0)
        assert g["status"].tolist() == o["status"].tolist() == [G.ST_MAXSTEPS, G.ST_CAPTURED, G.ST_NUMERIC, G.ST_OUTSIDE, G.ST_OUTSIDE]
        assert np.array_equal(g["steps_done"], o["steps_done"])
        assert parity.rel_err(g["final_state"], o["final_state"]).max() <= 1e-9
        assert parity.rel_err(g["health"], o["health"]).max() <= 1e-6
    rng = np.random.default_rng(7)
    m = 200
    out = np.array([np.log(rng.uniform(5, 40, m)), rng.uniform(0.3, 2.8, m), np.zeros(m), rng.uniform(5, 60, m),
                    rng.uniform(-3, 3, m), rng.uniform(-3, 3, m)])
    o = tab_oracle.integrate(tb, out, 0.05, 20000, nthreads=NCPU)
    g = run_gpu_tab(G, tb, out, 0.05, 20000)
    assert_parity(g, o, 1e-9)
    assert (g["status"] == G.ST_OUTSIDE).sum() > m // 2


def test_tabulated_empty_and_argument_errors(G):
    import torch
    tb = W.kerr_metric_table(1.0, 0.5, 65, 33, 3.0, 20.0, 0.3, math.pi - 0.3)
    ctx = G.geo_create_tabulated(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    dev = torch.device("cuda:0")
    out = G.alloc_outputs(0, dev)
    G.geo_integrate(ctx, torch.empty((6, 0), dtype=torch.float64, device=dev), 0.01, 10, out)     # n = 0: no-op
    st = torch.from_numpy(W.kerr_bound(8, 0.5, W.SEED_BASE + 4)).to(dev)
    for bad_flags in (G.FLAG_CARTESIAN_SNAP, G.FLAG_STAGED_SNAP):      # records exist on this path, but only the direct BL-style writer
        with pytest.raises(G.GeoError) as ei:
            G.geo_integrate(ctx, st, 0.01, 10, G.alloc_outputs(8, dev, 10, 5), snapshot_every=5, flags=bad_flags)
        assert ei.value.code == G.EINVAL
    with pytest.raises(G.GeoError) as ei:
        G.geo_integrate(ctx, st, 0.01, 10, G.alloc_outputs(8, dev), flags=G.FLAG_STATIC_MAP)
    assert ei.value.code == G.EINVAL
    with pytest.raises(G.GeoError) as ei:          # the adaptive path exists for five-field tables (T7), without flags
        G.geo_integrate_adaptive(ctx, st, 0.01, 1e-9, 1e-9, 100, G.alloc_outputs(8, dev, 0, 1, 4), snap_dtau=1.0, flags=G.FLAG_CARTESIAN_SNAP)
    assert ei.value.code == G.EINVAL
    assert math.isnan(G.geo_horizon_radius(ctx))
    G.geo_destroy(ctx)
    for bad in (dict(d1=0.0), dict(d2=-1.0), dict(x1_0=float("nan"))):
        kw = dict(x1_0=tb["x1_0"], d1=tb["d1"], x2_0=tb["x2_0"], d2=tb["d2"])
        kw.update(bad)
        with pytest.raises(G.GeoError):
            G.geo_create_tabulated(tb["tab"], **kw)
    with pytest.raises(G.GeoError):
        G.geo_create_tabulated(np.ones((5, 3, 8)), 0.0, 1.0, 0.0, 1.0)          # n2 < 4


def test_flat_space_straight_lines_on_the_gpu(G):
    """No oracle: Minkowski space in spherical coordinates, motion in the plane theta = pi/2 where the tabulated
    metric is exact (quadratic r^2; sin^2 = 1 with zero gradient on a grid line) -- the CUDA path must follow
    x(tau) = x0 + u tau, t = sqrt(1 + u^2) tau to RK4 accuracy."""
    n1, n2 = 47, 33
    d1, d2 = 11.5 / (n1 - 1), math.pi / (n2 - 1)
    x1 = 0.5 + d1 * (np.arange(n1 + 4) - 2)
    x2 = d2 * (np.arange(n2 + 4) - 2)
    R, TH = np.meshgrid(x1, x2)
    tb = {"tab": np.ascontiguousarray(np.stack([np.ones_like(R), np.zeros_like(R), np.ones_like(R), R * R, R * R * np.sin(TH) ** 2])),
          "x1_0": float(x1[0]), "d1": d1, "x2_0": float(x2[0]), "d2": d2}
    rng = np.random.default_rng(8)
    m = 500
    x0 = rng.uniform(-4, 4, (2, m))
    x0[0] += np.where(x0[0] > 0, 2.5, -2.5)          # keep |x| > 2.5 so the line stays away from r < 0.5 ... mostly
    u = rng.uniform(-0.5, 0.5, (2, m))
    r0 = np.hypot(x0[0], x0[1])
    st = np.array([r0, np.full(m, math.pi / 2), np.arctan2(x0[1], x0[0]), (x0 * u).sum(axis=0) / r0, np.zeros(m),
                   x0[0] * u[1] - x0[1] * u[0]])
    g = run_gpu_tab(G, tb, st, 0.01, 400)
    ok = g["status"] == G.ST_MAXSTEPS
    assert ok.mean() > 0.8
    xe = x0 + 4.0 * u
    r, th, ph, E = g["final_state"][1], g["final_state"][2], g["final_state"][3], g["final_state"][4]
    assert np.abs(th[ok] - math.pi / 2).max() < 1e-12
    assert np.abs(E[ok] - np.sqrt(1 + (u * u).sum(axis=0))[ok]).max() < 1e-14
    assert np.abs(r * np.cos(ph) - xe[0])[ok].max() < 1e-8 and np.abs(r * np.sin(ph) - xe[1])[ok].max() < 1e-8
    assert np.abs(g["final_state"][0] - 4.0 * E)[ok].max() < 1e-11


def test_tabulated_kerr_converges_to_the_analytic_kernel(G):
    """No oracle: the tabulated-metric kernel on eq.(8) tables of increasing resolution against the analytic-metric
    kernel (geo_rk4_kernel) on the same orbits -- the difference falls at least like the square of the grid spacing."""
    from gpu_helpers import run_gpu
    a = 0.9
    st = W.kerr_bound(2000, a, W.SEED_BASE + 2)
    ref = run_gpu(G, G.KERR, a, st, 0.01, 1500)
    res = []
    for n1, n2 in ((513, 129), (2049, 513)):
        tb = W.kerr_metric_table(1.0, a, n1, n2, 1.8, 40.0, 0.2, math.pi - 0.2)
        res.append(run_gpu_tab(G, tb, st, 0.01, 1500))
    ok = (res[0]["status"] == G.ST_MAXSTEPS) & (res[1]["status"] == G.ST_MAXSTEPS)     # the rest left the theta range
    assert ok.mean() > 0.9
    rows = [0, 1, 2, 3, 5, 6]
    errs = [parity.rel_err(g["final_state"][rows][:, ok], ref["final_state"][rows][:, ok]).max() for g in res]
    assert errs[1] < 1e-4 and errs[0] / errs[1] > 6, errs


@pytest.mark.parametrize("host,flags,mask,cap", [(False, 0, 0xFF, None), (False, 16, 0x0F, None), (True, 0, 0x26, 4), (False, 1, 0x07, 4)])
def test_tabulated_trajectory_records(G, tab_oracle, host, flags, mask, cap):
    """Records on the tabulated path (round 2; readings S1-S3 with the table's own coordinates): against the oracle,
    device and host entry points, stencil-cache and gather kernels, plain update, odd masks, capacity overflow; and slot j
    equals the final state of the run that stops there, bitwise."""
    import torch
    a = 0.9
    tb = W.kerr_metric_table(1.0, a, 513, 129, 1.8, 40.0, 0.2, math.pi - 0.2)
    st = W.kerr_bound(1501, a, W.SEED_BASE + 2)
    o = tab_oracle.integrate(tb, st, 0.01, 1500, flags=flags & 1, snapshot_every=250, snap_capacity=cap, snap_mask=mask, nthreads=NCPU)
    ctx = G.geo_create_tabulated(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    try:
        n = st.shape[1]
        if host:
            out = G.alloc_outputs_host(n, 1500, 250, cap, mask)
            G.geo_integrate_host(ctx, np.ascontiguousarray(st), 0.01, 1500, out, flags=flags, snapshot_every=250)
        else:
            out = G.alloc_outputs(n, torch.device("cuda:0"), 1500, 250, cap, mask)
            G.geo_integrate(ctx, torch.from_numpy(st).cuda(), 0.01, 1500, out, flags=flags, snapshot_every=250)
            torch.cuda.synchronize()
        g = G.to_numpy(out)
        assert_parity(g, o, 1e-9)
        assert np.array_equal(g["snap_count"], o["snap_count"]) and (g["snap_count"] == 7).all()
        assert parity.snapshot_err(g, o).max() <= 1e-9
        capn = o["snapshots"].shape[1]
        valid = np.arange(capn)[None, :] < np.minimum(g["snap_count"], capn)[:, None]
        assert np.isnan(g["snapshots"][~valid]).all() and np.isfinite(g["snapshots"][valid]).all()
        if mask == 0xFF and not host:
            for j in (2, 6):
                oj = G.alloc_outputs(n, torch.device("cuda:0"))
                G.geo_integrate(ctx, torch.from_numpy(st).cuda(), 0.01, 250 * j, oj, flags=flags)
                torch.cuda.synchronize()
                assert np.array_equal(g["snapshots"][:, j, :], G.to_numpy(oj)["final_state"].T)
    finally:
        G.geo_destroy(ctx)


def _run_tab_adaptive(G, tb, st, h0, rtol, atol, max_attempts, host=False, snap_dtau=0.0, cap=0, mask=0xFF, **kw):
    import torch
    ctx = G.geo_create_tabulated(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    try:
        n = st.shape[1]
        if host:
            out = G.alloc_outputs_host(n, 0, 1 if snap_dtau else 0, cap, mask)
            rej = np.full(n, -1, dtype=np.int32)
            G.geo_integrate_adaptive_host(ctx, np.ascontiguousarray(st), h0, rtol, atol, max_attempts, out, rejected=rej, snap_dtau=snap_dtau, **kw)
            g = G.to_numpy(out)
            g["rejected"] = rej
            return g
        dev = torch.device("cuda:0")
        out = G.alloc_outputs(n, dev, 0, 1 if snap_dtau else 0, cap, mask)
        rej = torch.full((n,), -1, dtype=torch.int32, device=dev)
        G.geo_integrate_adaptive(ctx, torch.from_numpy(np.ascontiguousarray(st)).to(dev), h0, rtol, atol, max_attempts, out,
                                 rejected=rej, snap_dtau=snap_dtau, **kw)
        torch.cuda.synchronize()
        g = G.to_numpy(out)
        g["rejected"] = rej.cpu().numpy()
        return g
    finally:
        G.geo_destroy(ctx)


def test_tabulated_adaptive_fixed_step_mode_and_records(G, tab_oracle):
    """Reading T7 with the controller off (rtol = inf): identical step sequences, so final states and dense-output records
    must agree like the RK4 path's (1e-9); host entry point bitwise equal to the device one."""
    a = 0.9
    tb = W.kerr_metric_table(1.0, a, 513, 129, 1.8, 40.0, 0.2, math.pi - 0.2)
    st = W.kerr_bound(1501, a, W.SEED_BASE + 2)
    kw = dict(tau_end=40.0)
    o = tab_oracle.integrate_adaptive(tb, st, 0.05, np.inf, 1.0, 10**6, snap_dtau=0.7, snap_capacity=60, nthreads=NCPU, **kw)
    g = _run_tab_adaptive(G, tb, st, 0.05, float("inf"), 1.0, 10**6, snap_dtau=0.7, cap=60, **kw)
    assert_parity(g, o, 1e-9)
    done = g["status"] == G.ST_MAXSTEPS              # a few orbits leave the table's theta range early (OUTSIDE): fewer records
    assert (g["rejected"] == 0).all() and np.array_equal(g["snap_count"], o["snap_count"])
    assert (g["snap_count"][done] == 1 + int(40.0 / 0.7)).all() and done.mean() > 0.95
    assert parity.snapshot_err(g, o).max() <= 1e-9
    gh = _run_tab_adaptive(G, tb, st, 0.05, float("inf"), 1.0, 10**6, host=True, snap_dtau=0.7, cap=60, **kw)
    for k in ("final_state", "status", "steps_done", "snapshots", "snap_count", "rejected"):
        assert np.array_equal(g[k], gh[k], equal_nan=True), k


def test_tabulated_adaptive_step_control_rays_and_domain_exit(G, tab_oracle):
    """Step control on: log-radial camera rays (capture / escape) and particles that run off the table (OUTSIDE), class
    against the oracle; states at a common final time within the integrator's tolerance; accept/reject counts identical
    for nearly all."""
    a = 0.998
    rp = W.horizon_radius(1.0, a)
    tb = W.kerr_metric_table(1.0, a, 1025, 257, math.log(0.005), math.log(80.0), 0.02, math.pi - 0.02, radial="log")
    full = W.camera_rays(64, a, 60.0, r_obs=50.0)
    st = W.to_log_radial(np.ascontiguousarray(full[:, ::5]), rp)
    kw = dict(r_capture=math.log(0.01), r_escape=math.log(55.0 - rp), kind=G.NULL)
    okw = dict(r_capture=math.log(0.01), r_escape=math.log(55.0 - rp), kind=tab_oracle.NULL)
    o = tab_oracle.integrate_adaptive(tb, st, 0.02, 1e-9, 1e-9, 100000, nthreads=NCPU, **okw)
    g = _run_tab_adaptive(G, tb, st, 0.02, 1e-9, 1e-9, 100000, **kw)
    assert np.array_equal(g["status"], o["status"]) and set(np.unique(g["status"])) >= {G.ST_CAPTURED, G.ST_ESCAPED}
    # The interpolated metric is only C^1: the error estimate jumps at every cell face, steps are rejected there, and whether
    # an attempt next to a face passes depends on the last bits -- the accept/reject SEQUENCES of the two sides differ for
    # almost every ray (unlike on the analytic metrics).  What is unique: the class, the amount of work to a few per cent,
    # and the state at a common final time (below, and for the rays at tau = 40 before any of them ends).
    work_g, work_o = g["steps_done"] + g["rejected"], o["steps_done"] + o["rejected"]
    assert abs(work_g.sum() / work_o.sum() - 1.0) < 0.05
    o40 = tab_oracle.integrate_adaptive(tb, st, 0.02, 1e-10, 1e-10, 100000, tau_end=40.0, nthreads=NCPU, **okw)
    g40 = _run_tab_adaptive(G, tb, st, 0.02, 1e-10, 1e-10, 100000, tau_end=40.0, **kw)
    assert np.array_equal(g40["status"], o40["status"]) and (g40["status"] == G.ST_MAXSTEPS).all()
    e40 = parity.rel_err(g40["final_state"], o40["final_state"]).max(axis=0)
    # ... and that state is only as well defined as the method is accurate on a C^1 metric: two step sequences that both
    # satisfy the controller differ by the error the kinks at the cell faces inject (the estimate does not see it in
    # full).  The oracle measures it on itself (rtol 1e-10 against 1e-11); the CUDA path must agree with the oracle to within
    # a small multiple of that, i.e. as well as the oracle agrees with itself.
    o40b = tab_oracle.integrate_adaptive(tb, st, 0.02, 1e-11, 1e-11, 100000, tau_end=40.0, nthreads=NCPU, **okw)
    d_self = parity.rel_err(o40["final_state"], o40b["final_state"]).max(axis=0)
    print("tab adaptive rays at tau = 40: max err", e40.max(), "oracle rtol 1e-10 vs 1e-11:", d_self.max())
    assert e40.max() <= max(5.0 * d_self.max(), 1e-7) and e40.max() <= 1e-4
    # bound orbits to a common final time; a few leave the table's theta range: OUTSIDE on both sides
    a2 = 0.9
    tb2 = W.kerr_metric_table(1.0, a2, 513, 129, 1.8, 40.0, 0.4, math.pi - 0.4)
    st2 = W.kerr_bound(2001, a2, W.SEED_BASE + 2)
    o2 = tab_oracle.integrate_adaptive(tb2, st2, 0.05, 1e-11, 1e-11, 10**6, tau_end=150.0, nthreads=NCPU)
    g2 = _run_tab_adaptive(G, tb2, st2, 0.05, 1e-11, 1e-11, 10**6, tau_end=150.0)
    assert np.array_equal(g2["status"], o2["status"])
    assert (g2["status"] == G.ST_OUTSIDE).any() and (g2["status"] == G.ST_MAXSTEPS).mean() > 0.8
    done = g2["status"] == G.ST_MAXSTEPS
    e = parity.rel_err(g2["final_state"], o2["final_state"]).max(axis=0)
    print("tab adaptive: OUTSIDE", int((g2["status"] == G.ST_OUTSIDE).sum()), "max err at tau_end", e[done].max(), "p99", np.quantile(e[done], 0.99))
    o2b = tab_oracle.integrate_adaptive(tb2, st2, 0.05, 1e-12, 1e-12, 10**6, tau_end=150.0, nthreads=NCPU)
    d2 = parity.rel_err(o2["final_state"], o2b["final_state"]).max(axis=0)[done & (o2b["status"] == tab_oracle.ST_MAXSTEPS)]
    print("   oracle rtol 1e-11 vs 1e-12: p99", np.quantile(d2, 0.99), "max", d2.max())
    assert np.quantile(e[done], 0.99) <= max(5.0 * np.quantile(d2, 0.99), 1e-7) and e[done].max() <= max(5.0 * d2.max(), 1e-6)
