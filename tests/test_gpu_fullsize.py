"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (persistent
grid, work queue on, same flags), on SAMPLED outputs the oracle can compute one by one.

Geodesics are independent, so the oracle run of a sampled particle alone must equal that
particle's entry in the full batch.  Samples are seeded; tolerances are the north_star's (1e-9 timelike,
1e-8 + class identity for certified null rays, readings P2/P3).  Beyond the samples, properties
that hold at any size are checked over the whole batch: constants of motion bit-exact, health |2H+kappa|
small, every particle terminated with a legal status / step count.
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


def _run_full(G, a, st, h, nsteps, snapshot_every=0, snap_mask=0xFF, **stop):
    import torch
    dev = torch.device("cuda:0")
    ctx = G.geo_create(G.KERR, 1.0, a)
    try:
        d_in = torch.from_numpy(st).to(dev)
        out = G.alloc_outputs(st.shape[1], dev, nsteps, snapshot_every, None, snap_mask)
        G.geo_integrate(ctx, d_in, h, nsteps, out, snapshot_every=snapshot_every, **stop)
        torch.cuda.synchronize()
        return out
    finally:
        G.geo_destroy(ctx)


def _take(out, ii, with_snaps=False):
    """Sampled entries of the device-resident outputs as numpy (the snapshot buffer can be > host RAM)."""
    import torch
    it = torch.from_numpy(ii).to(out["final_state"].device)
    g = {"final_state": out["final_state"][:, it].cpu().numpy(), "status": out["status"][it].cpu().numpy(),
         "steps_done": out["steps_done"][it].cpu().numpy(), "eq_cross_r": out["eq_cross_r"][it].cpu().numpy(),
         "health": out["health"][it].cpu().numpy()}
    if with_snaps:
        g["snapshots"] = out["snapshots"][it].cpu().numpy()
        g["snap_count"] = out["snap_count"][it].cpu().numpy()
    return g


def _sample(n, m, seed):
    rng = np.random.default_rng(seed)
    ii = np.unique(np.concatenate([[0, 1, n - 2, n - 1], rng.integers(0, n, size=m)]))
    return ii.astype(np.int64)


def test_config4_full_2p22_sampled(G, oracle):
    """configs[3], the bench workload: Kerr a=0.5, 2^22 bound timelike particles x 10^4 steps."""
    a, n = 0.5, 1 << 22
    st = W.kerr_bound(n, a, W.SEED_BASE + 4, nthreads=NCPU, chunk=1 << 20)
    out = _run_full(G, a, st, 0.01, 10000)
    assert int(out["status"].ne(G.ST_MAXSTEPS).sum().item()) == 0
    assert int(out["steps_done"].ne(10000).sum().item()) == 0
    hl = out["health"].cpu().numpy()
    assert np.quantile(hl, 0.9999) < 1e-9 and np.isfinite(hl).all()     # 2H + 1 drift is O(h^4) (DESIGN.md pins)
    fs = out["final_state"]
    assert bool((fs[7].cpu() == __import__("torch").from_numpy(st[5])).all())     # L = p_phi bit-exact (eq.(13))
    ii = _sample(n, 100_000, 41)          # ~9.5e4 distinct particles x 10^4 steps = 1e9 oracle steps (~10 s on the box)
    g = _take(out, ii)
    o = oracle.integrate(oracle.KERR, 1.0, a, np.ascontiguousarray(st[:, ii]), 0.01, 10000, nthreads=NCPU)
    c = parity.compare(g, o)
    print(f"config 4: {len(ii)} sampled particles vs oracle: max err {c['err'].max():.3e}, p99.9 {np.quantile(c['err'], 0.999):.3e}")
    assert len(ii) >= 90_000
    assert c["same_class"].all()
    assert c["err"].max() <= 1e-9, c["err"].max()


def test_config2_full_65536_sampled(G, oracle):
    """configs[1]: Kerr a=0.9, 65 536 bound particles x 10^5 steps, snapshot every 1000 (101 slots x 8)."""
    a, n = 0.9, 65536
    st = W.kerr_bound(n, a, W.SEED_BASE + 2, nthreads=NCPU)
    out = _run_full(G, a, st, 0.01, 100000, snapshot_every=1000)
    assert int(out["status"].ne(G.ST_MAXSTEPS).sum().item()) == 0
    assert int(out["snap_count"].ne(101).sum().item()) == 0
    ii = _sample(n, 4096, 42)             # ~4e3 particles x 10^5 steps = 4e8 oracle steps
    g = _take(out, ii, with_snaps=True)
    o = oracle.integrate(oracle.KERR, 1.0, a, np.ascontiguousarray(st[:, ii]), 0.01, 100000,
                         snapshot_every=1000, nthreads=NCPU)
    # reading P3: every particle the oracle itself determines to 1e-10 (double vs long double) must be within 1e-9,
    # final record AND all 101 trajectory records; the others (low-|L_z| orbits that pass next to the polar axis, reading
    # B7) are counted and printed.  Round 1 compared 160 particles and met none of them.
    def certify(jj):
        sub = np.ascontiguousarray(st[:, ii[jj]])
        kw = dict(snapshot_every=1000, nthreads=NCPU)
        return [oracle.integrate(oracle.KERR, 1.0, a, sub, 0.01, 100000, long_double=True, **kw),
                oracle.integrate(oracle.KERR, 1.0, a, parity.ulp_nudged(sub), 0.01, 100000, **kw)]
    rep = parity.p3_report(g, o, certify, 1e-9, labels=st[[0, 1, 3, 4, 5]][:, ii], max_fail_frac=0.002,
                           what="config 2 (labels: r0, theta0, u_r, u_theta, L_z)",
                           extra_err=parity.snapshot_err(g, o), extra_err_fn=parity.snapshot_err)
    print(f"config 2: {len(ii)} sampled particles incl. 101 records each vs oracle: {rep}")
    assert len(ii) >= 3800 and rep["class_mismatch"] == 0


def _escapes_analytic(a, Lz, Q, r_plus, r_obs):
    """Exact class of an incoming E = 1 photon: it escapes iff the radial potential
    R(r) = r^4 + (a^2 - L^2 - Q) r^2 + 2[Q + (L-a)^2] r - a^2 Q has a turning point in (r_+, r_obs).  Since
    R(r_+) = [(r_+^2 + a^2) - aL]^2 >= 0 and R(r_obs) > 0, that is: R <= 0 at an interior critical point
    (roots of the cubic R')."""
    c2 = a * a - Lz * Lz - Q
    c1 = 2.0 * (Q + (Lz - a) ** 2)
    c0 = -a * a * Q
    roots = W._cubic_real_roots(np.full_like(Lz, 4.0), np.zeros_like(Lz), 2.0 * c2, c1)
    esc = np.zeros(Lz.shape, dtype=bool)
    for k in range(3):
        rk = roots[k]
        Rk = ((rk * rk + c2) * rk + c1) * rk + c0
        with np.errstate(invalid="ignore"):
            esc |= (rk > r_plus) & (rk < r_obs) & (Rk <= 0.0)
    return esc


def _critical_band(esc_img, px):
    """Pixels within +-px (Chebyshev) of the analytic critical curve = the boundary between the escaping and the
    captured region of the image: those that have both classes in their (2 px + 1)^2 neighbourhood."""
    def dilate(m):
        out = m.copy()
        for _ in range(px):
            q = out.copy()
            q[1:, :] |= out[:-1, :]; q[:-1, :] |= out[1:, :]
            out = q.copy()
            q[:, 1:] |= out[:, :-1]; q[:, :-1] |= out[:, 1:]
            out = q
        return out
    return dilate(esc_img) & dilate(~esc_img)


def _null_oracle(oracle, st, a, ii, long_double=False, snapshot_every=0, snap_mask=0xFF, nudge=False):
    sub = np.ascontiguousarray(st[:, ii])
    return oracle.integrate(oracle.KERR, 1.0, a, parity.ulp_nudged(sub) if nudge else sub, 0.02, 200000,
                            r_capture=W.horizon_radius(1.0, a) + 0.01, r_escape=1100.0, kind=oracle.NULL,
                            snapshot_every=snapshot_every, snap_mask=snap_mask, long_double=long_double, nthreads=NCPU)


def _null_sets_vs_oracle(G, oracle, st, consts, a, out, sets, snapshot_every=0, snap_mask=0xFF, cert_stat=600):
    """Compare the rays of every named index set with the oracle under reading P3 (tests/parity.py:
    null_parity_report).  Returns {name: report}.  A fixed sub-sample of the first set also gets the long double oracle
    unconditionally, for the certified-fraction statistic DESIGN.md quotes."""
    reports = {}
    for name, ii in sets.items():
        if len(ii) == 0:
            continue
        o = _null_oracle(oracle, st, a, ii, snapshot_every=snapshot_every, snap_mask=snap_mask)
        g = _take(out, ii, with_snaps=snapshot_every > 0)
        skw = dict(snapshot_every=snapshot_every, snap_mask=snap_mask)
        rep = parity.p3_report(
            g, o, lambda jj: [_null_oracle(oracle, st, a, ii[jj], long_double=True, **skw),
                              _null_oracle(oracle, st, a, ii[jj], nudge=True, **skw)],
            1e-8, labels=consts[:, ii], max_fail_frac=0.10 if name in ("axis", "band") else 0.03, what=name,
            extra_err=parity.snapshot_err(g, o) if snapshot_every > 0 else None,            # trajectories: same bar
            extra_err_fn=parity.snapshot_err if snapshot_every > 0 else None)
        print(f"{name}: {rep}")
        reports[name] = rep
    first = next(iter(sets))
    jj = sets[first][:cert_stat]
    if len(jj):
        o0 = _null_oracle(oracle, st, a, jj)
        cert = (parity.certified(o0, _null_oracle(oracle, st, a, jj, long_double=True), 1e-8)
                & parity.certified(o0, _null_oracle(oracle, st, a, jj, nudge=True), 1e-8))
        print(f"certified fraction on {len(jj)} rays of '{first}': {cert.mean():.4f}")
        assert cert.mean() > 0.97
    return reports


def test_config3_full_1024x1024_vs_oracle_at_a_resolution_that_can_fail(G, oracle):
    """configs[2]: a=0.998, i=60 deg, the whole 1024^2 image in one call (work queue refilling lanes as rays are
    captured / escape).  north_star: class identical on >= 99.99 % of pixels, 1e-8 on the rest -- asserted where it can
    fail (round-1 verdict, 'what's weak' 1):
      * every pixel against the closed-form capture/escape criterion (no oracle): mismatches only in the axis columns;
      * 12 000 uniformly sampled pixels against the oracle: at most one class mismatch (99.99 %), all certified rays 1e-8;
      * EVERY pixel within +-3 px of the analytic critical curve and EVERY pixel of the 10 columns next to the polar axis
        (reading B7) against the oracle: all certified rays identical in class and within 1e-8, the others counted and
        printed with (alpha, beta, L_z, Q) (reading P3);
      * image-level class bar: (mismatches in band + axis, counted exhaustively) + 0 in the uniform sample of the rest
        <= 1e-4 x 2^20 pixels."""
    a, N = 0.998, 1024
    st, consts = W.camera_rays(N, a, 60.0, return_constants=True)
    al, be, Lz, Q = consts
    rp = W.horizon_radius(1.0, a)
    out = _run_full(G, a, st, 0.02, 200000, r_capture=rp + 0.01, r_escape=1100.0, kind=G.NULL)
    status = out["status"].cpu().numpy()
    counts = np.bincount(status, minlength=4)
    assert counts[G.ST_NUMERIC] == 0
    assert counts[G.ST_MAXSTEPS] <= 1e-3 * N * N          # only near-axis garbage rays hit the cap (B7)
    assert 0.15 < counts[G.ST_CAPTURED] / (N * N) < 0.25
    # closed form, all pixels
    esc = _escapes_analytic(a, Lz, Q, rp, 1000.0)
    wrong = (status == G.ST_ESCAPED) != esc
    axis = np.abs(al) < 0.1                      # the 10 pixel columns around alpha = 0
    print("closed-form class mismatches:", int(wrong.sum()), "of which in the axis columns:", int((wrong & axis).sum()),
          "captured fraction analytic / gpu:", float((~esc).mean()), float((status == G.ST_CAPTURED).mean()))
    assert (wrong & ~axis).sum() <= 8             # measured: 0
    assert wrong.sum() <= 2e-3 * N * N
    health = out["health"].cpu().numpy()
    if (wrong & axis).any():
        assert np.median(health[wrong & axis]) > 1e-9     # flagged as numerically invalid
    # oracle, at a resolution that can fail
    band = _critical_band(esc.reshape(N, N), 3).ravel() & ~axis
    rest = np.flatnonzero(~band & ~axis)
    rng = np.random.default_rng(43)
    sets = {"uniform": np.sort(rng.choice(rest, 12000, replace=False)), "band": np.flatnonzero(band), "axis": np.flatnonzero(axis)}
    print({k: len(v) for k, v in sets.items()})
    assert len(sets["band"]) > 5000 and len(sets["axis"]) == 10 * N
    rep = _null_sets_vs_oracle(G, oracle, st, consts, a, out, sets)
    assert rep["uniform"]["class_mismatch"] <= 1          # 99.99 % of 12 000
    # image-level literal bar: band and axis columns are counted exhaustively, the rest has (at most) the sampled rate
    est = rep["band"]["class_mismatch"] + rep["axis"]["class_mismatch"] + rep["uniform"]["class_mismatch"] * len(rest) / 12000.0
    print(f"class (status AND steps_done) mismatches: band {rep['band']['class_mismatch']} of {rep['band']['n']}, axis "
          f"{rep['axis']['class_mismatch']} of {rep['axis']['n']}, uniform {rep['uniform']['class_mismatch']} of 12000 -> image-level "
          f"estimate {est:.0f} of {N * N} pixels ({100.0 * (1 - est / (N * N)):.4f} % identical)")
    assert est <= 1e-4 * N * N


def test_config5_whole_4096x4096_image_in_16_tiles(G, oracle):
    """configs[4] as specified: i=85 deg, the WHOLE 4096^2 image, snapshot every 500 steps of (t, r, theta, phi) -- the
    dense trajectory buffer at the step cap is 215 GB > HBM, so the harness walks 16 tiles of 256 rows (reading S3;
    13.5 GB of records per tile, one buffer reused).  Per tile: every pixel against the closed-form capture/escape
    criterion, S1 (snap_count = 1 + steps_done // 500) on every ray; against the oracle (final record AND trajectory,
    reading P3): the stride-16 sub-image, every pixel within +-3 px of the analytic critical curve, and every 16th row
    of the 40 columns next to the polar axis."""
    import torch
    a, N, rows, every = 0.998, 4096, 256, 500
    rp = W.horizon_radius(1.0, a)
    dev = torch.device("cuda:0")
    ctx = G.geo_create(G.KERR, 1.0, a)
    n = N * rows
    out = G.alloc_outputs(n, dev, 200000, every, None, 0x0F)
    tot = {"steps": 0, "records": 0, "wrong": 0, "wrong_off_axis": 0, "captured": 0, "maxsteps": 0}
    agg = {}
    try:
        for t in range(N // rows):
            row0 = t * rows
            lo, hi = max(0, row0 - 3), min(N, row0 + rows + 3)                 # 3-row halo for the critical band
            st_h, c_h = W.camera_rays(N, a, 85.0, row0=lo, rows=hi - lo, return_constants=True)
            sl = slice((row0 - lo) * N, (row0 - lo) * N + n)
            st, consts = np.ascontiguousarray(st_h[:, sl]), c_h[:, sl]
            al = consts[0]
            G.geo_integrate(ctx, torch.from_numpy(st).to(dev), 0.02, 200000, out, snapshot_every=every,
                            r_capture=rp + 0.01, r_escape=1100.0, kind=G.NULL)
            torch.cuda.synchronize()
            status = out["status"].cpu().numpy()
            sd = out["steps_done"].cpu().numpy()
            sc = out["snap_count"].cpu().numpy()
            assert np.isin(status, (G.ST_MAXSTEPS, G.ST_CAPTURED, G.ST_ESCAPED)).all()
            assert np.array_equal(sc, 1 + sd // every)                           # S1 at any size
            esc_h = _escapes_analytic(a, c_h[2], c_h[3], rp, 1000.0)
            esc = esc_h[sl]
            wrong = (status == G.ST_ESCAPED) != esc
            axis = np.abs(al) < 0.1                                              # 40 columns around alpha = 0
            tot["steps"] += int(sd.sum()); tot["records"] += int(sc.sum())
            tot["wrong"] += int(wrong.sum()); tot["wrong_off_axis"] += int((wrong & ~axis).sum())
            tot["captured"] += int((status == G.ST_CAPTURED).sum()); tot["maxsteps"] += int((status == G.ST_MAXSTEPS).sum())
            band = _critical_band(esc_h.reshape(hi - lo, N), 3).ravel()[sl] & ~axis
            img = np.arange(n).reshape(rows, N)
            stride = img[8::16, 8::16].ravel()
            stride = stride[~band[stride] & ~axis[stride]]
            ax = img[8::16, :].ravel()
            sets = {"stride16": stride, "band": np.flatnonzero(band), "axis": ax[axis[ax]]}
            rep = _null_sets_vs_oracle(G, oracle, st, consts, a, out, sets, snapshot_every=every, snap_mask=0x0F,
                                       cert_stat=100 if t in (0, 7) else 0)
            for k, r in rep.items():
                d = agg.setdefault(k, {"n": 0, "class_mismatch": 0, "fail": 0})
                for q in d:
                    d[q] += r[q]
            print(f"tile {t}: classes captured {int((status == G.ST_CAPTURED).sum())} escaped {int((status == G.ST_ESCAPED).sum())} "
                  f"cap {int((status == G.ST_MAXSTEPS).sum())}; closed-form mismatches {int(wrong.sum())} (off axis {int((wrong & ~axis).sum())})")
    finally:
        G.geo_destroy(ctx)
    npx = N * N
    print(f"config 5 whole image: {tot['steps']:.4e} geodesic-steps, {tot['records']} records = {tot['records'] * 32 / 1e9:.1f} GB written "
          f"(dense buffer would be {npx * 401 * 32 / 1e9:.0f} GB), captured {tot['captured'] / npx:.4f}, at the step cap {tot['maxsteps']}, "
          f"closed-form class mismatches {tot['wrong']} (off the axis columns: {tot['wrong_off_axis']}); vs oracle: {agg}")
    assert tot["wrong_off_axis"] <= 64 and tot["wrong"] <= 5e-3 * npx
    assert 0.10 < tot["captured"] / npx < 0.25
    assert agg["stride16"]["n"] > 60000 and agg["band"]["n"] > 20000 and agg["axis"]["n"] >= 10000
    assert agg["stride16"]["class_mismatch"] <= max(1, int(1e-4 * agg["stride16"]["n"]))      # 99.99 % on the regular sub-image


def test_tab4_full_2p22_tabulated_sampled(G, tab_oracle):
    """bench.py --workload tab4: the 2^22 particles of configs[3] through the 2053 x 517-node table of
    the Kerr a = 0.5 metric, 1000 steps, in the bench's launch configuration; sampled particles against the
    tabulated-metric oracle, whole-batch properties."""
    import math
    import torch
    a, n = 0.5, 1 << 22
    st = W.kerr_bound(n, a, W.SEED_BASE + 4, nthreads=NCPU, chunk=1 << 20)
    tb = W.kerr_metric_table(1.0, a, 2049, 513, 2.0, 45.0, 0.1, math.pi - 0.1)
    dev = torch.device("cuda:0")
    ctx = G.geo_create_tabulated(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    try:
        out = G.alloc_outputs(n, dev)
        G.geo_integrate(ctx, torch.from_numpy(st).to(dev), 0.01, 1000, out)
        torch.cuda.synchronize()
    finally:
        G.geo_destroy(ctx)
    ii = _sample(n, 3000, 11)
    g = _take(out, ii)
    o = tab_oracle.integrate(tb, np.ascontiguousarray(st[:, ii]), 0.01, 1000, nthreads=NCPU)
    c = parity.compare(g, o)
    assert c["same_class"].all() and c["err"].max() <= 1e-9, c["err"].max()
    status = out["status"].cpu().numpy()
    assert np.isin(status, (G.ST_MAXSTEPS, G.ST_OUTSIDE)).all() and (status == G.ST_MAXSTEPS).mean() > 0.99
    assert np.array_equal(out["final_state"][7].cpu().numpy(), st[5])            # p_phi exact
    assert np.nanmax(out["health"].cpu().numpy()) < 1e-6


def test_config3a_full_image_adaptive_sampled(G, oracle):
    """bench.py --workload config3a: all 1024^2 rays of configs[2] with the adaptive stepper; sampled
    rays against the oracle's adaptive path: class identical, the escaped photon's direction and momenta within 1e-8 on
    certified rays (see below for what a fixed tolerance leaves undetermined)."""
    import torch
    a, N = 0.998, 1024
    st = W.camera_rays(N, a, 60.0)
    rc = W.horizon_radius(1.0, a) + 0.01
    dev = torch.device("cuda:0")
    ctx = G.geo_create(G.KERR, 1.0, a)
    try:
        out = G.alloc_outputs(N * N, dev)
        rej = torch.zeros(N * N, dtype=torch.int32, device=dev)
        G.geo_integrate_adaptive(ctx, torch.from_numpy(st).to(dev), 0.02, 1e-9, 1e-9, 200000, out, r_capture=rc,
                                 r_escape=1100.0, kind=G.NULL, rejected=rej)
        torch.cuda.synchronize()
    finally:
        G.geo_destroy(ctx)
    ii = _sample(N * N, 3000, 12)
    g = _take(out, ii)
    grej = rej[torch.from_numpy(ii).to(dev)].cpu().numpy()
    kw = dict(r_capture=rc, r_escape=1100.0, kind=oracle.NULL, nthreads=NCPU)
    sub = np.ascontiguousarray(st[:, ii])
    o = oracle.integrate_adaptive(oracle.KERR, 1.0, a, sub, 0.02, 1e-9, 1e-9, 200000, **kw)
    o_ld = oracle.integrate_adaptive(oracle.KERR, 1.0, a, sub, 0.02, 1e-9, 1e-9, 200000, long_double=True, **kw)
    assert (g["status"] == o["status"]).mean() >= 0.999
    # What is unique at a fixed tolerance: the controller's error estimate is a difference of nearly equal numbers, so
    # its rounding noise (~1e-8 relative in h, measured between the oracle's double and long double runs) moves the
    # point ALONG the ray at which an escaping ray is stopped (t, r: ~1e-7 relative), while the ray itself -- theta,
    # phi, p_r, p_theta of the escaped photon -- is fixed to ~1e-11.  Reading P3 carried over to those components: a
    # ray is certified iff the oracle's double and long double runs agree in class and within 1e-9 on them.  Captured
    # rays: class only (their record is the last accepted state next to the horizon).
    rows = [2, 3, 5, 6]
    esc = o["status"] == oracle.ST_ESCAPED
    cert = esc & (o_ld["status"] == o["status"]) & (parity.rel_err(o["final_state"][rows], o_ld["final_state"][rows]).max(axis=0) <= 1e-9)
    e_ray = parity.rel_err(g["final_state"][rows], o["final_state"][rows]).max(axis=0)
    e_along = parity.rel_err(g["final_state"][[0, 1]], o["final_state"][[0, 1]]).max(axis=0)
    same = (g["status"] == o["status"]) & (g["steps_done"] == o["steps_done"]) & (grej == o["rejected"])
    print("adaptive full image: escaped", esc.mean(), "certified", cert.mean(), "same sequence", same.mean(),
          "max err on certified: ray", e_ray[cert].max(), "along", e_along[cert].max())
    assert cert.sum() > 0.9 * esc.sum() and same.mean() >= 0.95
    assert (g["status"] == o["status"])[cert].all()
    assert e_ray[cert].max() <= 1e-8 and e_along[cert].max() <= 1e-6, (e_ray[cert].max(), e_along[cert].max())


def test_config3a_full_image_adaptive_dense_records_cover_captured_rays_too(G, oracle):
    """Round-1 verdict ('what's weak' 4): at full image size the adaptive path's CAPTURED rays were compared by class only,
    because their final record is the last accepted state, and where that lies depends on the step-size noise.  With
    dense output (reading A3) every ray -- captured or escaped -- has records at the SAME affine times tau_j = 100 j on
    both sides: all 1024^2 rays are traced with records, 6000 sampled rays (captured ones over-sampled) are compared record
    by record at 1e-8 under reading P3, and the number of records may differ by at most the last one."""
    import torch
    a, N = 0.998, 1024
    st, consts = W.camera_rays(N, a, 60.0, return_constants=True)
    rc = W.horizon_radius(1.0, a) + 0.01
    dev = torch.device("cuda:0")
    cap, dtau = 24, 100.0
    ctx = G.geo_create(G.KERR, 1.0, a)
    try:
        out = G.alloc_outputs(N * N, dev, 0, 1, cap, 0x6F)              # t, r, theta, phi, p_r, p_theta
        rej = torch.zeros(N * N, dtype=torch.int32, device=dev)
        G.geo_integrate_adaptive(ctx, torch.from_numpy(st).to(dev), 0.02, 1e-9, 1e-9, 200000, out, r_capture=rc,
                                 r_escape=1100.0, kind=G.NULL, rejected=rej, snap_dtau=dtau)
        torch.cuda.synchronize()
    finally:
        G.geo_destroy(ctx)
    status = out["status"].cpu().numpy()
    rng = np.random.default_rng(14)
    ii = np.sort(np.concatenate([rng.choice(np.flatnonzero(status == G.ST_CAPTURED), 3000, replace=False),
                                 rng.choice(np.flatnonzero(status == G.ST_ESCAPED), 3000, replace=False)]))
    g = _take(out, ii, with_snaps=True)
    kw = dict(r_capture=rc, r_escape=1100.0, kind=oracle.NULL, nthreads=NCPU, snap_dtau=dtau, snap_capacity=cap, snap_mask=0x6F)

    def run(sub, **extra):
        return oracle.integrate_adaptive(oracle.KERR, 1.0, a, np.ascontiguousarray(sub), 0.02, 1e-9, 1e-9, 200000, **kw, **extra)
    o = run(st[:, ii])
    assert np.array_equal(g["status"], o["status"])
    assert (np.abs(g["snap_count"].astype(int) - o["snap_count"]) <= 1).all()

    def common_records_err(x, y):
        """worst P2 error over the records BOTH runs produced (the last record may exist on one side only)."""
        m = np.minimum(np.minimum(x["snap_count"], y["snap_count"]), cap)
        valid = np.arange(cap)[None, :] < m[:, None]
        return np.where(valid[:, :, None], parity.rel_err(x["snapshots"], y["snapshots"]), 0.0).max(axis=(1, 2))
    err = common_records_err(g, o)
    fail = np.flatnonzero(~(err <= 1e-8))
    print(f"adaptive dense records, {len(ii)} rays (3000 captured): max err {err.max():.3e}, outside 1e-8: {len(fail)}")
    assert len(fail) <= 0.03 * len(ii)
    if len(fail):                                                       # reading P3: they must be uncertified
        o_sub = parity.take(o, fail)
        cert = np.ones(len(fail), dtype=bool)
        for o_c in (run(st[:, ii[fail]], long_double=True), run(parity.ulp_nudged(st[:, ii[fail]]))):
            cert &= (o_c["status"] == o_sub["status"]) & (common_records_err(o_sub, o_c) <= 1e-9)
        for k, i in enumerate(fail[:12]):
            print(f"   ray {ii[i]} status {g['status'][i]} err {err[i]:.3e} certified {bool(cert[k])} (alpha, beta, Lz, Q) = {consts[:, ii[i]]}")
        assert not cert.any()
    captured = g["status"] == G.ST_CAPTURED
    assert (g["snap_count"][captured] >= 10).all()                      # ~1000 M of affine time to the hole: >= 10 records each
