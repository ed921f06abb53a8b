"""GPU parity of the Cartesian Kerr-Schild path (GEO_KERR_SCHILD, csrc/geo_ks.cuh; SURVEY 8(f).3 second clause, DESIGN.md
readings K1-K5) against its oracle (oracle/geo_ks_oracle.cpp), element by element on the same seeded inputs, through the
C ABI: bound orbits of the config-2 distribution (1e-9), camera rays of config 3 incl. the polar-axis columns (class
identity and 1e-8 under reading P3), trajectory records, particles through the polar axis and through the horizon, edge
cases, host entry point, static mapping; and -- no oracle involved -- the WHOLE config-3 image against the closed-form
capture criterion: the polar-axis columns that the Boyer-Lindquist path gets wrong (reading B7) come out right."""
import math
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import parity  # noqa: E402
from gpu_helpers import run_gpu, assert_snapshots_match  # noqa: E402
from test_gpu_fullsize import _escapes_analytic, _critical_band  # noqa: E402  (closed-form class of an E = 1 photon; no oracle)

from paper_1803_08320_b200 import workloads as W  # noqa: E402

pytestmark = pytest.mark.gpu
NCPU = max(1, (os.cpu_count() or 1))


def _orbits(n, a=0.9):
    st, consts = W.kerr_bound(n, a, W.SEED_BASE + 2, return_constants=True)
    return W.to_cartesian_kerr_schild(st, consts[0], 1.0, a), st, consts


@pytest.mark.parametrize("flags", [0, 1, 2])
def test_bound_orbits_parity(G, ks_oracle, flags):
    """3001 orbits (23 full CTAs + a ragged tail) x 4000 steps, Kerr a = 0.9: every output within 1e-9 of the oracle
    (reading P3 certification for the few that pass next to the axis); Kahan / plain update, queue / static mapping."""
    a = 0.9
    ks, st, consts = _orbits(3001, a)
    oflags = flags & 1
    o = ks_oracle.integrate(1.0, a, ks, 0.01, 4000, flags=oflags, nthreads=NCPU)
    g = run_gpu(G, G.KERR_SCHILD, a, ks, 0.01, 4000, flags=flags)
    rep = parity.p3_report(g, o, lambda jj: [ks_oracle.integrate(1.0, a, np.ascontiguousarray(ks[:, jj]), 0.01, 4000, flags=oflags, long_double=True),
                                             ks_oracle.integrate(1.0, a, parity.ulp_nudged(np.ascontiguousarray(ks[:, jj])), 0.01, 4000, flags=oflags)],
                           1e-9, labels=consts, max_fail_frac=0.002, what=f"Kerr-Schild bound orbits, flags {flags}")
    print(rep)
    assert rep["class_mismatch"] == 0
    ok = np.isfinite(o["health"])
    assert np.max(np.abs(g["health"][ok] - o["health"][ok])) < 1e-11
    # the chart's own check: L_z = x p_y - y p_x is NOT a momentum here; it must still be conserved to O(h^4)
    f = g["final_state"]
    assert np.max(np.abs(f[1] * f[6] - f[2] * f[5] - consts[1])) < 1e-7


def test_energy_matches_oracle_to_rounding(G, ks_oracle):
    ks, st, consts = _orbits(257, 0.9)
    g = run_gpu(G, G.KERR_SCHILD, 0.9, ks, 0.01, 0)
    E = np.array([ks_oracle.energy(1.0, 0.9, *ks[:, i], 1.0) for i in range(257)])
    assert np.max(np.abs(g["final_state"][4] - E) / E) < 1e-15
    assert np.max(np.abs(g["final_state"][4] - consts[0]) / consts[0]) < 1e-13    # = the Boyer-Lindquist E of the same covector


def test_host_entry_equals_device_path_bitwise(G):
    ks, _, _ = _orbits(1500, 0.9)
    kw = dict(snapshot_every=100, snap_mask=0x0F, r_capture=2.0, r_escape=28.0)
    d = run_gpu(G, G.KERR_SCHILD, 0.9, ks, 0.01, 1000, **kw)
    h = run_gpu(G, G.KERR_SCHILD, 0.9, ks, 0.01, 1000, host=True, **kw)
    for k in ("final_state", "status", "steps_done", "snap_count", "health"):
        assert np.array_equal(d[k], h[k], equal_nan=True), k
    assert np.array_equal(d["eq_cross_r"], h["eq_cross_r"], equal_nan=True)
    valid = np.arange(d["snapshots"].shape[1])[None, :] < d["snap_count"][:, None]
    assert np.array_equal(d["snapshots"][valid], h["snapshots"][valid])


@pytest.mark.parametrize("flags,mask,cap", [(0, 0xFF, None), (0, 0x0F, None), (1, 0x6E, None), (0, 0xFF, 4), (2, 0x81, 3)])
def test_trajectory_records(G, ks_oracle, flags, mask, cap):
    """Records (readings S1-S3) with the direct 256-bit writer and the masked fallback, capacity overflow; slot j bitwise
    equal to the GPU run that stops after j * snapshot_every steps."""
    a = 0.9
    ks, _, _ = _orbits(1201, a)
    kw = dict(r_capture=2.2, r_escape=27.0)
    o = ks_oracle.integrate(1.0, a, ks, 0.01, 1200, flags=flags & 1, snapshot_every=200, snap_capacity=cap, snap_mask=mask, nthreads=NCPU, **kw)
    g = run_gpu(G, G.KERR_SCHILD, a, ks, 0.01, 1200, flags=flags, snapshot_every=200, snap_capacity=cap, snap_mask=mask, **kw)
    assert np.array_equal(g["status"], o["status"]) and np.array_equal(g["steps_done"], o["steps_done"])
    assert len(np.unique(o["status"])) >= 2
    assert_snapshots_match(g, o, 1e-9)
    if cap is None:
        comps = [k for k in range(8) if (mask >> k) & 1]
        for j in (1, 4):
            s = run_gpu(G, G.KERR_SCHILD, a, ks, 0.01, 200 * j, flags=flags, **kw)
            ok = g["steps_done"] >= 200 * j
            assert ok.sum() > 1000
            assert np.array_equal(g["snapshots"][ok, j, :], s["final_state"][comps][:, ok].T)


def _camera(a, incl, N, sel):
    full, consts = W.camera_rays(N, a, incl, return_constants=True)
    st = np.ascontiguousarray(full[:, sel])
    ks = W.to_cartesian_kerr_schild(st, np.ones(st.shape[1]), 1.0, a)
    return ks, st, np.ascontiguousarray(consts[:, sel])


def test_camera_rays_parity_incl_axis_columns(G, ks_oracle, oracle):
    """configs[2] rays (a = 0.998, i = 60 deg, h = 0.02, capture at r_+ + 0.01, escape at 1100): a strided 32 x 32 sub-image
    and 64 rows of the 10 polar-axis columns.  Against the Kerr-Schild oracle: class (status AND steps_done) identical and
    1e-8 under reading P3.  Against the closed form: every ray off the +-3 px critical band correct -- also in the axis
    columns.  Against the
    Boyer-Lindquist oracle (another chart, another right-hand side): same class flag, r at the end within 1e-6 on the
    rays that are healthy there."""
    a, N = 0.998, 1024
    rp = W.horizon_radius(1.0, a)
    img = np.arange(N * N).reshape(N, N)
    consts_full = W.camera_rays(N, a, 60.0, return_constants=True)[1]
    esc_full = _escapes_analytic(a, consts_full[2], consts_full[3], rp, 1000.0)
    band_full = _critical_band(esc_full.reshape(N, N), 3).ravel()
    sub = img[16::32, 16::32].ravel()
    axis = img[8::16, N // 2 - 5:N // 2 + 5].ravel()
    for name, sel in (("sub-image", sub), ("axis columns", axis)):
        ks, st, consts = _camera(a, 60.0, N, sel)
        kw = dict(r_capture=rp + 0.01, r_escape=1100.0)
        o = ks_oracle.integrate(1.0, a, ks, 0.02, 200000, kind=ks_oracle.NULL, nthreads=NCPU, **kw)
        g = run_gpu(G, G.KERR_SCHILD, a, ks, 0.02, 200000, kind=G.NULL, **kw)
        rep = parity.p3_report(
            g, o, lambda jj: [ks_oracle.integrate(1.0, a, np.ascontiguousarray(ks[:, jj]), 0.02, 200000, kind=ks_oracle.NULL, long_double=True, nthreads=NCPU, **kw),
                              ks_oracle.integrate(1.0, a, parity.ulp_nudged(np.ascontiguousarray(ks[:, jj])), 0.02, 200000, kind=ks_oracle.NULL, nthreads=NCPU, **kw)],
            1e-8, labels=consts, max_fail_frac=0.03, what=f"Kerr-Schild camera rays, {name}")
        print(name, rep, "classes", np.bincount(g["status"], minlength=4).tolist(), "max health", float(g["health"].max()))
        assert rep["class_mismatch"] <= max(1, int(1e-4 * len(sel)))
        esc = esc_full[sel]
        off_band = ~band_full[sel]
        # closed form: no wrong pixel off the +-3 px band of the critical curve -- the polar-axis columns included
        assert np.array_equal((g["status"] == G.ST_ESCAPED)[off_band], esc[off_band]), name
        assert set(np.unique(g["status"])) <= {G.ST_CAPTURED, G.ST_ESCAPED}
        escaped = g["status"] == G.ST_ESCAPED
        print("   health of escaped rays: median %.1e max %.1e" % (np.median(g["health"][escaped]), g["health"][escaped].max()))
        assert np.median(g["health"][escaped]) < 1e-13
        if name == "axis columns":
            assert g["health"][escaped].max() < 1e-8         # the Boyer-Lindquist path: up to 1e47 here (reading B7)
        # the Boyer-Lindquist oracle on the same rays
        ob = oracle.integrate(oracle.KERR, 1.0, a, st, 0.02, 200000, kind=oracle.NULL, nthreads=NCPU, **kw)
        healthy = ob["health"] < 1e-9
        assert np.array_equal(g["status"][healthy], ob["status"][healthy])
        r_ks = W.kerr_schild_radius(g["final_state"][1:4], a)
        cth = g["final_state"][3] / r_ks
        e2 = healthy & (g["status"] == G.ST_ESCAPED) & (g["steps_done"] == ob["steps_done"])
        if name == "sub-image":          # (in the axis columns NO ray is healthy in Boyer-Lindquist coordinates: nothing to compare)
            assert healthy.sum() > 0.7 * len(sel) and e2.sum() > 0.5 * healthy.sum()
            assert np.max(np.abs(r_ks[e2] - ob["final_state"][1][e2]) / 1100.0) < 1e-6
            assert np.max(np.abs(cth[e2] - np.cos(ob["final_state"][2][e2]))) < 1e-6
        if name == "axis columns":
            print("Boyer-Lindquist oracle: unhealthy axis rays", int((~healthy).sum()), "of", len(sel),
                  "wrong class there:", int(((ob["status"] == oracle.ST_ESCAPED) != esc).sum()))


def test_whole_config3_image_closed_form_and_oracle_at_a_resolution_that_can_fail(G, ks_oracle):
    """The whole 1024^2 image of configs[2] in ONE call on the Kerr-Schild path (work queue on).
    (1) Every pixel against the closed-form capture / escape criterion.  The 10 polar-axis columns, where the
    Boyer-Lindquist path has its 533 wrong pixels and |2H| up to 1e47 (reading B7), come out right: 0 mismatches, |2H| < 1e-8.
    What this chart pays: next to the prograde photon orbit of a = 0.998 (r = 1.074 M, 0.01 M outside the horizon) the
    Cartesian components turn by ~0.75 rad per step of h = 0.02 M, and <= 64 pixels (measured: 42; 10 at h = 0.01) within
    3 px of the prograde edge of the shadow are captured instead of escaping -- on the GPU and in the oracle alike
    (DESIGN.md section 8.5).  No ray at the step cap.
    (2) Against the oracle, the north_star's null-ray rule where it can fail (reading P3): 6000 uniformly sampled pixels,
    EVERY pixel within +-3 px of the analytic critical curve, EVERY pixel of the axis columns -- class (status AND
    steps_done) identical on >= 99.99 %, 1e-8 on every certified ray, the others counted and printed."""
    import torch
    a, N = 0.998, 1024
    rp = W.horizon_radius(1.0, a)
    st, consts = W.camera_rays(N, a, 60.0, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, np.ones(N * N), 1.0, a)
    dev = torch.device("cuda:0")
    kw = dict(r_capture=rp + 0.01, r_escape=1100.0)
    ctx = G.geo_create(G.KERR_SCHILD, 1.0, a)
    try:
        out = G.alloc_outputs(N * N, dev)
        G.geo_integrate(ctx, torch.from_numpy(ks).to(dev), 0.02, 200000, out, kind=G.NULL, **kw)
        torch.cuda.synchronize()
        g_all = G.to_numpy(out)
    finally:
        G.geo_destroy(ctx)
    status, health, steps = g_all["status"], g_all["health"], g_all["steps_done"]
    esc = _escapes_analytic(a, consts[2], consts[3], rp, 1000.0)
    wrong = (status == G.ST_ESCAPED) != esc
    counts = np.bincount(status, minlength=4)
    print("classes", counts.tolist(), "closed-form mismatches", int(wrong.sum()), "max health", float(health.max()),
          "steps total", int(steps.sum()))
    assert counts[G.ST_MAXSTEPS] == 0 and counts[G.ST_NUMERIC] == 0
    axis = np.abs(consts[0]) < 0.1                       # the 10 pixel columns around alpha = 0
    band = _critical_band(esc.reshape(N, N), 3).ravel()
    print("mismatches in the axis columns", int((wrong & axis).sum()), "off the +-3 px critical band", int((wrong & ~band).sum()),
          "L_z of the mismatching pixels", consts[2][wrong].min() if wrong.any() else None, consts[2][wrong].max() if wrong.any() else None)
    assert (wrong & axis).sum() == 0                     # the Boyer-Lindquist path: 533
    assert (wrong & ~band).sum() == 0
    assert wrong.sum() <= 64                             # measured: 42, the prograde edge of the shadow
    assert np.all(consts[2][wrong] > 1.9)
    escaped = status == G.ST_ESCAPED
    assert health[escaped & axis].max() < 1e-8 and np.median(health[escaped]) < 1e-13
    # (2) the oracle
    rest = np.flatnonzero(~band & ~axis)
    rng = np.random.default_rng(47)
    sets = {"uniform": np.sort(rng.choice(rest, 6000, replace=False)), "band": np.flatnonzero(band & ~axis), "axis": np.flatnonzero(axis)}
    print({k: len(v) for k, v in sets.items()})
    assert len(sets["band"]) > 5000 and len(sets["axis"]) == 10 * N

    def orc(ii, **extra):
        sub = np.ascontiguousarray(ks[:, ii])
        if extra.pop("nudge", False):
            sub = parity.ulp_nudged(sub)
        return ks_oracle.integrate(1.0, a, sub, 0.02, 200000, kind=ks_oracle.NULL, nthreads=NCPU, **kw, **extra)
    mism = {}
    for name, ii in sets.items():
        o = orc(ii)
        g = parity.take(g_all, ii)
        rep = parity.p3_report(g, o, lambda jj: [orc(ii[jj], long_double=True), orc(ii[jj], nudge=True)], 1e-8,
                               labels=consts[:, ii], max_fail_frac=0.03, what=f"Kerr-Schild image, {name}")
        print(name, rep)
        mism[name] = rep["class_mismatch"]
    assert mism["uniform"] == 0
    est = mism["band"] + mism["axis"] + mism["uniform"] * len(rest) / 6000.0
    print(f"class mismatches: band {mism['band']}, axis {mism['axis']}, uniform {mism['uniform']} -> image-level estimate {est:.0f} of {N * N}")
    assert est <= 1e-4 * N * N


def test_ks4_full_2p22_sampled(G, ks_oracle):
    """The bench workload `ks4` at FULL size in the launch configuration bench.py times (2^22 config-4 particles in Cartesian
    Kerr-Schild coordinates x 2500 steps, persistent grid, queue on): 20 000 sampled particles against the oracle at 1e-9;
    over the whole batch every particle ends with MAXSTEPS after 2500 steps, E bit-equal to the zero-step run's, |2H + 1| small."""
    import torch
    a, n = 0.5, 1 << 22
    st, consts = W.kerr_bound(n, a, W.SEED_BASE + 4, nthreads=NCPU, chunk=1 << 20, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, consts[0], 1.0, a)
    dev = torch.device("cuda:0")
    ctx = G.geo_create(G.KERR_SCHILD, 1.0, a)
    try:
        out = G.alloc_outputs(n, dev)
        G.geo_integrate(ctx, torch.from_numpy(ks).to(dev), 0.01, 2500, out)
        torch.cuda.synchronize()
        assert bool((out["status"] == G.ST_MAXSTEPS).all()) and bool((out["steps_done"] == 2500).all())
        assert float(out["health"].max()) < 1e-9
        g_all = G.to_numpy(out)
    finally:
        G.geo_destroy(ctx)
    f = g_all["final_state"]
    assert np.max(np.abs(f[4] - consts[0]) / consts[0]) < 1e-13                      # E: constant, = the Boyer-Lindquist E
    assert np.max(np.abs(f[1] * f[6] - f[2] * f[5] - consts[1])) < 1e-8              # L_z conserved by the dynamics, O(h^4)
    rng = np.random.default_rng(53)
    ii = np.unique(np.concatenate([[0, 1, n - 2, n - 1], rng.integers(0, n, size=20000)])).astype(np.int64)
    sub = np.ascontiguousarray(ks[:, ii])
    o = ks_oracle.integrate(1.0, a, sub, 0.01, 2500, nthreads=NCPU)
    rep = parity.p3_report(parity.take(g_all, ii), o,
                           lambda jj: [ks_oracle.integrate(1.0, a, np.ascontiguousarray(sub[:, jj]), 0.01, 2500, long_double=True),
                                       ks_oracle.integrate(1.0, a, parity.ulp_nudged(np.ascontiguousarray(sub[:, jj])), 0.01, 2500)],
                           1e-9, labels=consts[:, ii], max_fail_frac=0.001, what="ks4 sampled")
    print(f"ks4: {len(ii)} sampled particles vs oracle: {rep}")
    assert rep["class_mismatch"] == 0 and len(ii) > 19000


def test_through_the_polar_axis_and_through_the_horizon(G, ks_oracle):
    """Where eq.(8) divides by sin^2(theta) or Delta: particles aimed through x = y = 0 and particles followed to 0.9 r_+
    (inside the hole).  1e-9 against the oracle, all of them; the infallers end inside r_+ with finite state."""
    for a in (0.9, 0.998):
        rp = W.horizon_radius(1.0, a)
        n = 96
        st = np.zeros((6, n))
        for k in range(48):
            st[:, k] = [-6.0, 0.0 if k % 2 == 0 else 1e-7 * k, 7.0 + 0.1 * k, 1.2, 0.0, 0.01 * (k % 7)]
        for k in range(48, n):
            j = k - 48
            st[:, k] = [7.0 + 0.05 * j, 1.0, 0.1 * (j - 20), -0.4, 0.004 * j, 0.0]
        kw = dict(r_capture=0.9 * rp, r_escape=200.0)
        o = ks_oracle.integrate(1.0, a, st, 0.01, 6000, nthreads=NCPU, **kw)
        g = run_gpu(G, G.KERR_SCHILD, a, st, 0.01, 6000, **kw)
        c = parity.compare(g, o)
        print(f"a = {a}: classes {np.bincount(g['status'], minlength=4).tolist()} max err {c['err'].max():.2e}")
        assert c["same_class"].all() and c["err"].max() <= 1e-9
        inside = g["status"] == G.ST_CAPTURED
        assert inside[48:].all() and not inside[:48].any()
        assert np.all(W.kerr_schild_radius(g["final_state"][1:4, inside], a) < rp) and np.isfinite(g["final_state"]).all()


def test_edge_cases_and_argument_errors(G, ks_oracle):
    import torch
    a = 0.9
    ks, _, _ = _orbits(40, a)
    ks[0:3, 0] = [0.3, 0.2, 0.5]         # inside r_capture
    ks[0:3, 1] = [300.0, 0.0, 50.0]      # beyond r_escape
    ks[4, 2] = np.nan                    # non-finite momentum
    ks[0:3, 3] = [0.0, 0.0, 5.0]         # ON the polar axis
    kw = dict(r_capture=1.5, r_escape=100.0, snapshot_every=5)
    o = ks_oracle.integrate(1.0, a, ks, 0.01, 20, **kw)
    g = run_gpu(G, G.KERR_SCHILD, a, ks, 0.01, 20, **kw)
    assert np.array_equal(g["status"], o["status"]) and np.array_equal(g["steps_done"], o["steps_done"])
    assert g["status"][0] == G.ST_CAPTURED and g["status"][1] == G.ST_ESCAPED and g["status"][2] == G.ST_NUMERIC
    assert g["status"][3] == G.ST_MAXSTEPS and np.isfinite(g["final_state"][:, 3]).all()
    assert np.array_equal(g["snap_count"], o["snap_count"]) and g["snap_count"][0] == 0 and g["snap_count"][1] == 1
    ok = np.ones(40, bool)
    ok[2] = False
    assert parity.rel_err(g["final_state"], o["final_state"])[:, ok].max() <= 1e-12
    # backwards in tau, disabled stop radii, nsteps = 0
    for h, ns in ((-0.01, 300), (0.01, 0)):
        o = ks_oracle.integrate(1.0, a, ks[:, 4:], h, ns)
        g = run_gpu(G, G.KERR_SCHILD, a, ks[:, 4:], h, ns)
        c = parity.compare(g, o)
        assert c["same_class"].all() and c["err"].max() <= 1e-10
    # n = 0; unsupported flags
    ctx = G.geo_create(G.KERR_SCHILD, 1.0, a)
    try:
        d_in = torch.empty((6, 0), dtype=torch.float64, device="cuda:0")
        G.geo_integrate(ctx, d_in, 0.01, 10, G.alloc_outputs(0, d_in.device))
        d_in = torch.from_numpy(ks).to("cuda:0")
        out = G.alloc_outputs(40, d_in.device, 20, 5)
        for bad in (G.FLAG_CARTESIAN_SNAP, G.FLAG_STAGED_SNAP, G.FLAG_TAB_GATHER):
            with pytest.raises(Exception):
                G.geo_integrate(ctx, d_in, 0.01, 20, out, flags=bad, snapshot_every=5)
        with pytest.raises(Exception):       # the adaptive path exists in this chart (reading K6) but takes no flags
            G.geo_integrate_adaptive(ctx, d_in, 0.01, 1e-9, 1e-9, 1000, G.alloc_outputs(40, d_in.device), flags=G.FLAG_PLAIN_UPDATE)
        assert G.geo_horizon_radius(ctx) == pytest.approx(1.0 + math.sqrt(1.0 - a * a))
    finally:
        G.geo_destroy(ctx)
    with pytest.raises(Exception):
        G.geo_create(G.KERR_SCHILD, 1.0, 1.5)


# ---- reading K6: the adaptive RK5(4) stepper in this chart (geo_ks_rk45_kernel) -------------------------------------------
def _run_ks_adaptive(G, a, st, h0, rtol, atol, max_attempts, host=False, snap_dtau=0.0, cap=0, mask=0xFF, **kw):
    import torch
    ctx = G.geo_create(G.KERR_SCHILD, 1.0, a)
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


def test_adaptive_fixed_step_mode_step_control_and_records(G, ks_oracle):
    """(i) Controller off (rtol = inf): identical step sequences -- final states and dense-output records of 1501 orbits
    (ragged) to tau = 40 within 1e-9, odd mask and capacity overflow included; host entry bitwise equal to the device one.
    (ii) Controller on (rtol = atol = 1e-12, tau_end = 60): on this analytic metric the accept / reject sequences of the two
    sides agree for nearly every orbit, and the states at the common final time agree to 1e-9."""
    a = 0.9
    ks, st, consts = _orbits(1501, a)
    for mask, cap in ((0xFF, 60), (0x2E, 7)):
        o = ks_oracle.integrate_adaptive(1.0, a, ks, 0.05, np.inf, 1.0, 10**6, tau_end=40.0, snap_dtau=0.7, snap_capacity=cap, snap_mask=mask, nthreads=NCPU)
        g = _run_ks_adaptive(G, a, ks, 0.05, float("inf"), 1.0, 10**6, tau_end=40.0, snap_dtau=0.7, cap=cap, mask=mask)
        c = parity.compare(g, o)
        print("KS adaptive, controller off: max err", c["err"].max(), "records", parity.snapshot_err(g, o).max())
        assert c["same_class"].all() and c["err"].max() <= 1e-9
        assert (g["rejected"] == 0).all() and (g["steps_done"] == 800).all()
        assert np.array_equal(g["snap_count"], o["snap_count"]) and (g["snap_count"] == 1 + int(40.0 / 0.7)).all()
        assert parity.snapshot_err(g, o).max() <= 1e-9
    gh = _run_ks_adaptive(G, a, ks, 0.05, float("inf"), 1.0, 10**6, host=True, tau_end=40.0, snap_dtau=0.7, cap=7, mask=0x2E)
    for k in ("final_state", "status", "steps_done", "snapshots", "snap_count", "rejected"):
        assert np.array_equal(g[k], gh[k], equal_nan=True), k
    o = ks_oracle.integrate_adaptive(1.0, a, ks, 0.05, 1e-12, 1e-12, 10**6, tau_end=60.0, nthreads=NCPU)
    g = _run_ks_adaptive(G, a, ks, 0.05, 1e-12, 1e-12, 10**6, tau_end=60.0)
    assert np.array_equal(g["status"], o["status"]) and (g["status"] == G.ST_MAXSTEPS).all()
    same = (g["steps_done"] == o["steps_done"]) & (g["rejected"] == o["rejected"])
    e = parity.rel_err(g["final_state"], o["final_state"]).max(axis=0)
    print("KS adaptive, step control: same sequence", same.mean(), "max err at tau_end", e.max(), "mean accepted", g["steps_done"].mean())
    assert same.mean() >= 0.95 and e.max() <= 1e-9


def test_adaptive_whole_config3_image_every_pixel_class_right(G, ks_oracle):
    """The whole 1024^2 image of configs[2] with per-ray step control in this chart (rtol = atol = 1e-9): EVERY pixel's class
    equals the closed form -- the polar-axis columns where the fixed-step Boyer-Lindquist path has 533 wrong pixels AND the
    prograde edge of the shadow where the fixed-step path of this chart has 42 (readings K6a, K6b).  3000 sampled rays + every
    pixel of the axis columns' 64 sampled rows against the oracle: class identical; the escaped photon's momenta (constant
    far from the hole in this chart) within 1e-8 on the rays the oracle determines to 1e-9 (double vs long double), its
    position within 1e-6 (the stopping point moves along the ray with the controller's rounding noise)."""
    import torch
    a, N = 0.998, 1024
    rp = W.horizon_radius(1.0, a)
    st, consts = W.camera_rays(N, a, 60.0, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, np.ones(N * N), 1.0, a)
    dev = torch.device("cuda:0")
    kw = dict(r_capture=rp + 0.01, r_escape=1100.0)
    ctx = G.geo_create(G.KERR_SCHILD, 1.0, a)
    try:
        out = G.alloc_outputs(N * N, dev)
        rej = torch.zeros(N * N, dtype=torch.int32, device=dev)
        d_in = torch.from_numpy(ks).to(dev)
        G.geo_integrate_adaptive(ctx, d_in, 0.02, 1e-9, 1e-9, 200000, out, kind=G.NULL, rejected=rej, **kw)
        torch.cuda.synchronize()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        G.geo_integrate_adaptive(ctx, d_in, 0.02, 1e-9, 1e-9, 200000, out, kind=G.NULL, rejected=rej, **kw)
        t1.record()
        torch.cuda.synchronize()
        g_all = G.to_numpy(out)
        g_all["rejected"] = rej.cpu().numpy()
    finally:
        G.geo_destroy(ctx)
    status = g_all["status"]
    esc = _escapes_analytic(a, consts[2], consts[3], rp, 1000.0)
    wrong = (status == G.ST_ESCAPED) != esc
    work = g_all["steps_done"] + g_all["rejected"]
    print("KS adaptive image:", t0.elapsed_time(t1), "ms; classes", np.bincount(status, minlength=4).tolist(), "closed-form mismatches", int(wrong.sum()),
          "attempts per ray mean / max", work.mean(), work.max(), "max |2H| of escaped rays", g_all["health"][status == G.ST_ESCAPED].max())
    assert set(np.unique(status)) <= {G.ST_CAPTURED, G.ST_ESCAPED}
    assert wrong.sum() == 0
    assert g_all["health"][status == G.ST_ESCAPED].max() < 1e-4 and np.median(g_all["health"][status == G.ST_ESCAPED]) < 1e-8
    img = np.arange(N * N).reshape(N, N)
    rng = np.random.default_rng(61)
    ii = np.unique(np.concatenate([rng.integers(0, N * N, 3000), img[8::16, N // 2 - 5:N // 2 + 5].ravel(), np.flatnonzero(
        _critical_band(esc.reshape(N, N), 1).ravel())[::7]]))
    sub = np.ascontiguousarray(ks[:, ii])
    okw = dict(kind=ks_oracle.NULL, nthreads=NCPU, **kw)
    o = ks_oracle.integrate_adaptive(1.0, a, sub, 0.02, 1e-9, 1e-9, 200000, **okw)
    o_ld = ks_oracle.integrate_adaptive(1.0, a, sub, 0.02, 1e-9, 1e-9, 200000, long_double=True, **okw)
    g = parity.take(g_all, ii)
    assert (g["status"] == o["status"]).mean() >= 0.9999
    rows = [5, 6, 7]
    e_o = o["status"] == ks_oracle.ST_ESCAPED
    cert = e_o & (o_ld["status"] == o["status"]) & (parity.rel_err(o["final_state"][rows], o_ld["final_state"][rows]).max(axis=0) <= 1e-9)
    e_ray = parity.rel_err(g["final_state"][rows], o["final_state"][rows]).max(axis=0)
    e_along = parity.rel_err(g["final_state"][[0, 1, 2, 3]], o["final_state"][[0, 1, 2, 3]]).max(axis=0)
    same = (g["status"] == o["status"]) & (g["steps_done"] == o["steps_done"]) & (g["rejected"] == o["rejected"])
    print("   vs oracle on", len(ii), "rays: escaped", e_o.mean(), "certified", cert.mean(), "same sequence", same.mean(),
          "max err on certified: momenta", e_ray[cert].max(), "position", e_along[cert].max())
    assert cert.sum() > 0.9 * e_o.sum() and same.mean() >= 0.9
    assert (g["status"] == o["status"])[cert].all()
    assert e_ray[cert].max() <= 1e-8 and e_along[cert].max() <= 1e-6
