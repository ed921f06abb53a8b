"""GPU parity of the GENERAL tabulated-metric path (reading T6; include/geo.h:
geo_create_tabulated_general) with its oracle (oracle/geo_tab_oracle.cpp: integrate_general), element by element on the
same seeded inputs, plus checks that need no oracle: the embedded eq.(8) table must give what the five-field kernel
gives, and Kerr in horizon-penetrating Kerr-Schild coordinates must carry particles through r_+."""
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


def run_tabg(G, tb, st, h, nsteps, host=False, general=True, **kw):
    import torch
    mk = G.geo_create_tabulated_general if general else G.geo_create_tabulated
    ctx = mk(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    try:
        n = st.shape[1]
        if host:
            out = G.alloc_outputs_host(n)
            G.geo_integrate_host(ctx, np.ascontiguousarray(st), h, nsteps, out, **kw)
            return G.to_numpy(out)
        dev = torch.device("cuda:0")
        out = G.alloc_outputs(n, dev)
        G.geo_integrate(ctx, torch.from_numpy(np.ascontiguousarray(st)).to(dev), h, nsteps, out, **kw)
        torch.cuda.synchronize()
        return G.to_numpy(out)
    finally:
        G.geo_destroy(ctx)


@pytest.mark.parametrize("flags", [0, 1, 16, 17])      # 1 = plain update, 16 = GEO_FLAG_TAB_GATHER (no stencil cache)
def test_embedded_eq8_table_matches_oracle_and_the_five_field_kernel(G, tab_oracle, flags):
    a = 0.9
    tb5 = W.kerr_metric_table(1.0, a, 513, 129, 1.8, 40.0, 0.2, math.pi - 0.2)
    tb10 = W.general_table_from_diagonal(tb5)
    st = W.kerr_bound(3001, a, W.SEED_BASE + 2)
    o = tab_oracle.integrate_general(tb10, st, 0.01, 2000, flags=flags & 1, nthreads=NCPU)
    g = run_tabg(G, tb10, st, 0.01, 2000, flags=flags)
    c = parity.compare(g, o)
    assert c["same_class"].all() and c["err"].max() <= 1e-9, c["err"].max()
    assert np.array_equal(g["final_state"][7], st[5])                           # p_phi exact
    if flags & 16:                      # the stencil cache changes where the values come from, not a single bit
        gc = run_tabg(G, tb10, st, 0.01, 2000, flags=flags & 1)
        for k in ("final_state", "status", "steps_done", "eq_cross_r", "health"):
            assert np.array_equal(g[k], gc[k], equal_nan=True), k
    g5 = run_tabg(G, tb5, st, 0.01, 2000, flags=flags, general=False)
    c5 = parity.compare(g, g5)
    assert c5["same_class"].all() and c5["err"].max() <= 1e-11, c5["err"].max()
    gh = run_tabg(G, tb10, st[:, :777], 0.01, 2000, flags=flags, host=True)
    for k in ("final_state", "status", "steps_done", "eq_cross_r", "health"):
        assert np.array_equal(g[k][..., :777], gh[k], equal_nan=True), k


def test_kerr_schild_bound_orbits_vs_oracle_and_boyer_lindquist_kernel(G, tab_oracle):
    """Kerr a = 0.9 in ingoing Kerr-Schild coordinates (beta^r != 0, gamma_r phi != 0) on a 1025 x 257 table: 1e-9 against
    the oracle over 5000 steps; and, with no oracle involved, r, theta, p_theta of the same orbits from the ANALYTIC
    Boyer-Lindquist kernel (geo_rk4_kernel) -- the two coordinate systems share them -- to the interpolation error."""
    import torch
    a, M = 0.9, 1.0
    st, consts = W.kerr_bound(3001, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_kerr_schild(st, consts[0], M, a)
    tb = W.kerr_schild_metric_table(M, a, 1025, 257, 1.2, 40.0, 0.15, math.pi - 0.15)
    o = tab_oracle.integrate_general(tb, ks, 0.01, 5000, nthreads=NCPU)
    g = run_tabg(G, tb, ks, 0.01, 5000)
    rep = parity.p3_report(g, o, lambda jj: [tab_oracle.integrate_general(tb, np.ascontiguousarray(ks[:, jj]), 0.01, 5000, long_double=True, nthreads=NCPU),
                                             tab_oracle.integrate_general(tb, parity.ulp_nudged(np.ascontiguousarray(ks[:, jj])), 0.01, 5000, nthreads=NCPU)],
                           1e-9, labels=st[[0, 1, 3, 4, 5]], max_fail_frac=0.002, what="Kerr-Schild bound orbits")
    print(rep)
    done = g["status"] == G.ST_MAXSTEPS          # a few orbits leave the table's theta range (T4): same class as the oracle
    assert rep["class_mismatch"] == 0 and np.isin(g["status"], (G.ST_MAXSTEPS, G.ST_OUTSIDE)).all() and done.mean() > 0.97
    assert np.abs(g["final_state"][4] - consts[0])[done].max() < 1e-6     # E of the interpolated metric's mass shell
    ctx = G.geo_create(G.KERR, M, a)
    out = G.alloc_outputs(st.shape[1], torch.device("cuda:0"))
    G.geo_integrate(ctx, torch.from_numpy(st).cuda(), 0.01, 5000, out)
    torch.cuda.synchronize()
    bl = G.to_numpy(out)
    G.geo_destroy(ctx)
    d = np.abs(g["final_state"][[1, 2, 6]] - bl["final_state"][[1, 2, 6]]).max(axis=0)[done]
    print("KS table vs analytic BL kernel: median", np.median(d), "max", d.max())
    assert np.median(d) < 1e-5 and np.quantile(d, 0.99) < 2e-3


def test_kerr_schild_table_carries_particles_and_photons_through_the_horizon(G, tab_oracle):
    """Horizon penetration: infalling particles and the captured camera rays of config 3 are followed to r = 1.25 M, INSIDE
    r_+ = 1.0632 M ... for a = 0.998 (1.4359 M for a = 0.9) -- with finite states and |2H + kappa| small -- where the
    Boyer-Lindquist path must stop outside (Delta = 0).  Class and final record against the oracle."""
    M = 1.0
    # (1) timelike plunge, a = 0.9
    a = 0.9
    rp = M + math.sqrt(M * M - a * a)
    n = 256
    fall = np.zeros((6, n))
    fall[0] = np.linspace(4.0, 9.0, n)
    fall[1] = np.linspace(0.6, 2.5, n)
    fall[4] = 0.3
    fall[5] = np.linspace(-1.0, 1.0, n)
    E = np.sqrt((1.0 - 2.0 * M * fall[0] / (fall[0] ** 2 + a * a * np.cos(fall[1]) ** 2)))   # rough; only p_r~ depends on it
    ks = W.to_kerr_schild(fall, E, M, a)
    tb = W.kerr_schild_metric_table(M, a, 1025, 257, 1.1, 40.0, 0.15, math.pi - 0.15)
    kw = dict(r_capture=1.25, r_escape=39.0)
    o = tab_oracle.integrate_general(tb, ks, 0.005, 40000, nthreads=NCPU, **kw)
    g = run_tabg(G, tb, ks, 0.005, 40000, **kw)
    c = parity.compare(g, o)
    inside = (g["status"] == G.ST_CAPTURED)
    print("plunging particles captured inside the horizon:", inside.sum(), "of", n, "max err", c["err"].max())
    assert inside.sum() > n // 2 and (g["final_state"][1][inside] < rp - 0.1).all()
    assert c["same_class"].all() and c["err"].max() <= 1e-9
    assert np.isfinite(g["final_state"]).all() and np.nanmax(g["health"][inside]) < 1e-6
    # (2) photons: a strided sub-image of config 3 (E = 1), a = 0.998, capture radius inside the horizon
    a = 0.998
    rp = M + math.sqrt(M * M - a * a)
    full, consts = W.camera_rays(1024, a, 60.0, r_obs=60.0, return_constants=True)
    ii = np.arange(1024 * 1024).reshape(1024, 1024)[250:774:21, 250:774:21].ravel()
    st = np.ascontiguousarray(full[:, ii])
    ks = W.to_kerr_schild(st, np.ones(len(ii)), M, a)
    tb = W.kerr_schild_metric_table(M, a, 2049, 257, 0.9, 64.0, 0.02, math.pi - 0.02)
    kw = dict(r_capture=1.0, r_escape=62.0, kind=G.NULL)
    okw = dict(r_capture=1.0, r_escape=62.0, kind=tab_oracle.NULL)
    o = tab_oracle.integrate_general(tb, ks, 0.02, 20000, nthreads=NCPU, **okw)
    g = run_tabg(G, tb, ks, 0.02, 20000, **kw)
    rep = parity.p3_report(g, o, lambda jj: [tab_oracle.integrate_general(tb, np.ascontiguousarray(ks[:, jj]), 0.02, 20000, long_double=True, nthreads=NCPU, **okw),
                                             tab_oracle.integrate_general(tb, parity.ulp_nudged(np.ascontiguousarray(ks[:, jj])), 0.02, 20000, nthreads=NCPU, **okw)],
                           1e-8, labels=consts[:, ii], max_fail_frac=0.05, what="Kerr-Schild photons")
    cap = g["status"] == G.ST_CAPTURED
    print(rep, "captured inside r_+:", cap.sum(), "escaped:", (g["status"] == G.ST_ESCAPED).sum(), "other:", (~cap & (g["status"] != G.ST_ESCAPED)).sum())
    # the record of a captured photon is its last accepted state before a stage point passed r_capture = 1.0 (B2): most
    # of them lie inside r_+ = 1.0632, all within one step's travel of it
    rc_fin = g["final_state"][1][cap]
    assert cap.sum() > 50 and np.median(rc_fin) < rp and (rc_fin < rp + 0.1).all() and (g["status"] == G.ST_ESCAPED).sum() > 50
    assert np.isfinite(g["final_state"]).all()
    assert rep["class_mismatch"] <= 1


def test_general_table_argument_errors(G):
    import torch
    tb = W.general_table_from_diagonal(W.kerr_metric_table(1.0, 0.5, 33, 17, 2.0, 20.0, 0.3, 2.8))
    with pytest.raises(ValueError):
        G.geo_create_tabulated_general(tb["tab"][:5].copy(), tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    with pytest.raises(G.GeoError):
        G.geo_create_tabulated_general(tb["tab"], tb["x1_0"], -1.0, tb["x2_0"], tb["d2"])
    ctx = G.geo_create_tabulated_general(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    try:
        assert math.isnan(G.geo_horizon_radius(ctx))
        st = torch.from_numpy(W.kerr_bound(8, 0.5, W.SEED_BASE + 4)).cuda()
        with pytest.raises(G.GeoError):         # records exist on this path, but not the staged / Cartesian writers
            G.geo_integrate(ctx, st, 0.01, 10, G.alloc_outputs(8, st.device, 10, 5), snapshot_every=5, flags=G.FLAG_CARTESIAN_SNAP)
        with pytest.raises(G.GeoError):
            G.geo_integrate(ctx, st, 0.01, 10, G.alloc_outputs(8, st.device), flags=G.FLAG_STATIC_MAP)
        with pytest.raises(G.GeoError):         # the adaptive path exists on this metric (T6 + T7) but takes no flags
            G.geo_integrate_adaptive(ctx, st, 0.01, 1e-9, 1e-9, 100, G.alloc_outputs(8, st.device), flags=G.FLAG_CARTESIAN_SNAP)
    finally:
        G.geo_destroy(ctx)


@pytest.mark.parametrize("flags,mask,cap", [(0, 0xFF, None), (16, 0x0F, None), (1, 0x46, 3)])
def test_general_tabulated_trajectory_records(G, tab_oracle, flags, mask, cap):
    """Records on the general path (readings S1-S3) in Kerr-Schild coordinates: against the oracle, cache and gather
    kernels, plain update, odd mask, capacity overflow; slot j bitwise equal to the GPU run that stops there."""
    import torch
    a, M = 0.9, 1.0
    st, consts = W.kerr_bound(1201, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_kerr_schild(st, consts[0], M, a)
    tb = W.kerr_schild_metric_table(M, a, 513, 129, 1.2, 40.0, 0.15, math.pi - 0.15)
    o = tab_oracle.integrate_general(tb, ks, 0.01, 1200, flags=flags & 1, snapshot_every=200, snap_capacity=cap, snap_mask=mask, nthreads=NCPU)
    ctx = G.geo_create_tabulated_general(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    try:
        dev = torch.device("cuda:0")
        out = G.alloc_outputs(ks.shape[1], dev, 1200, 200, cap, mask)
        G.geo_integrate(ctx, torch.from_numpy(ks).to(dev), 0.01, 1200, out, flags=flags, snapshot_every=200)
        torch.cuda.synchronize()
        g = G.to_numpy(out)
        c = parity.compare(g, o)
        assert c["same_class"].all() and c["err"].max() <= 1e-9
        assert np.array_equal(g["snap_count"], o["snap_count"])
        assert parity.snapshot_err(g, o).max() <= 1e-9
        if mask == 0xFF:
            oj = G.alloc_outputs(ks.shape[1], dev)
            G.geo_integrate(ctx, torch.from_numpy(ks).to(dev), 0.01, 600, oj, flags=flags)
            torch.cuda.synchronize()
            done = g["snap_count"] > 3
            assert np.array_equal(g["snapshots"][done, 3, :], G.to_numpy(oj)["final_state"].T[done])
    finally:
        G.geo_destroy(ctx)


# ---- readings T6 + T7: the adaptive RK5(4) stepper on the general ten-field table ----------------------------------------
def _run_tabg_adaptive(G, tb, st, h0, rtol, atol, max_attempts, host=False, snap_dtau=0.0, cap=0, mask=0xFF, **kw):
    import torch
    ctx = G.geo_create_tabulated_general(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
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


def test_general_adaptive_fixed_step_mode_and_records(G, tab_oracle):
    """Controller off (rtol = inf): identical step sequences, so final states and dense-output records agree like the RK4
    path's (1e-9) -- Kerr a = 0.9 in Kerr-Schild coordinates, 1501 orbits (ragged) to tau = 40 with 58 records each, odd
    mask; host entry point bitwise equal to the device one."""
    a, M = 0.9, 1.0
    st, consts = W.kerr_bound(1501, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_kerr_schild(st, consts[0], M, a)
    tb = W.kerr_schild_metric_table(M, a, 513, 129, 1.2, 40.0, 0.15, math.pi - 0.15)
    for mask, cap in ((0xFF, 60), (0x2E, 7)):
        kw = dict(tau_end=40.0)
        o = tab_oracle.integrate_adaptive_general(tb, ks, 0.05, np.inf, 1.0, 10**6, snap_dtau=0.7, snap_capacity=cap, snap_mask=mask, nthreads=NCPU, **kw)
        g = _run_tabg_adaptive(G, tb, ks, 0.05, float("inf"), 1.0, 10**6, snap_dtau=0.7, cap=cap, mask=mask, **kw)
        c = parity.compare(g, o)
        print("general adaptive, controller off: max err", c["err"].max(), "records", parity.snapshot_err(g, o).max())
        assert c["same_class"].all() and c["err"].max() <= 1e-9
        done = g["status"] == G.ST_MAXSTEPS
        assert (g["rejected"] == 0).all() and np.array_equal(g["snap_count"], o["snap_count"])
        assert (g["snap_count"][done] == 1 + int(40.0 / 0.7)).all() and done.mean() > 0.95
        assert parity.snapshot_err(g, o).max() <= 1e-9
        ok = np.isfinite(o["health"])
        assert np.array_equal(np.isfinite(g["health"]), ok) and np.max(np.abs(g["health"][ok] - o["health"][ok])) < 1e-9
    gh = _run_tabg_adaptive(G, tb, ks, 0.05, float("inf"), 1.0, 10**6, host=True, snap_dtau=0.7, cap=7, mask=0x2E, **kw)
    for k in ("final_state", "status", "steps_done", "snapshots", "snap_count", "rejected"):
        assert np.array_equal(g[k], gh[k], equal_nan=True), k


def test_general_adaptive_step_control_plunge_and_domain_exit(G, tab_oracle):
    """Step control on, Kerr-Schild table: bound orbits to a common final time agree with the oracle as well as the oracle
    agrees with itself at a ten times tighter tolerance (the interpolant is C^1: accept / reject sequences differ, DESIGN.md
    8.2); particles thrown at the hole are followed through r_+ to the capture radius inside it (class identical); particles
    that run off the table end OUTSIDE on both sides."""
    a, M = 0.9, 1.0
    rp = M + math.sqrt(M * M - a * a)
    st, consts = W.kerr_bound(2001, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_kerr_schild(st, consts[0], M, a)
    tb = W.kerr_schild_metric_table(M, a, 513, 129, 1.2, 40.0, 0.3, math.pi - 0.3)
    o = tab_oracle.integrate_adaptive_general(tb, ks, 0.05, 1e-11, 1e-11, 10**6, tau_end=150.0, nthreads=NCPU)
    g = _run_tabg_adaptive(G, tb, ks, 0.05, 1e-11, 1e-11, 10**6, tau_end=150.0)
    assert np.array_equal(g["status"], o["status"])
    assert (g["status"] == G.ST_MAXSTEPS).mean() > 0.8
    done = g["status"] == G.ST_MAXSTEPS
    e = parity.rel_err(g["final_state"], o["final_state"]).max(axis=0)
    ob = tab_oracle.integrate_adaptive_general(tb, ks, 0.05, 1e-12, 1e-12, 10**6, tau_end=150.0, nthreads=NCPU)
    both = done & (ob["status"] == tab_oracle.ST_MAXSTEPS)
    d_self = parity.rel_err(o["final_state"], ob["final_state"]).max(axis=0)[both]
    work_g, work_o = g["steps_done"] + g["rejected"], o["steps_done"] + o["rejected"]
    print("general adaptive: OUTSIDE", int((g["status"] == G.ST_OUTSIDE).sum()), "max err at tau_end", e[done].max(), "p99", np.quantile(e[done], 0.99),
          "| oracle rtol 1e-11 vs 1e-12: p99", np.quantile(d_self, 0.99), "max", d_self.max(), "| work ratio", work_g.sum() / work_o.sum())
    assert np.quantile(e[done], 0.99) <= max(5.0 * np.quantile(d_self, 0.99), 1e-8) and e[done].max() <= max(5.0 * d_self.max(), 1e-6)
    assert abs(work_g.sum() / work_o.sum() - 1.0) < 0.05
    # plunge through the horizon
    tb2 = W.kerr_schild_metric_table(M, a, 1025, 257, 1.1, 40.0, 0.15, math.pi - 0.15)
    n = 256
    fall = np.zeros((6, n))
    fall[0] = np.linspace(4.0, 9.0, n)
    fall[1] = np.linspace(0.6, 2.5, n)
    fall[3] = -0.2
    fall[5] = np.linspace(-1.0, 1.0, n)
    kw = dict(r_capture=1.25, r_escape=39.0)
    o2 = tab_oracle.integrate_adaptive_general(tb2, fall, 0.05, 1e-9, 1e-9, 10**5, nthreads=NCPU, **kw)
    g2 = _run_tabg_adaptive(G, tb2, fall, 0.05, 1e-9, 1e-9, 10**5, **kw)
    assert np.array_equal(g2["status"], o2["status"]) and (g2["status"] == G.ST_CAPTURED).all()
    assert (g2["final_state"][1] >= 1.25).all() and (g2["final_state"][1] < rp).all() and np.isfinite(g2["final_state"]).all()
    assert np.nanmax(g2["health"]) < 1e-4
    # off the table
    out = ks[:, :300].copy()
    out[0] = 39.0
    out[3] = 2.0
    o3 = tab_oracle.integrate_adaptive_general(tb, out, 0.05, 1e-9, 1e-9, 10**5, nthreads=NCPU)
    g3 = _run_tabg_adaptive(G, tb, out, 0.05, 1e-9, 1e-9, 10**5)
    assert np.array_equal(g3["status"], o3["status"]) and (g3["status"] == G.ST_OUTSIDE).all()
    assert (g3["final_state"][1] <= 40.0).all()
