"""The large-angle path of the RK4 kernel against the oracle (round-1 verdict, 'what's weak' 3).

A step whose stage angle moves by |d| >= 2^-7 rad cannot use the angle-addition kernels of `stage_trig`; the lane then
discards the step's sum and recomputes it with a full sin/cos at every stage point (`rk4_sum_full`).
That path runs only next to the horizon or with a coarse h, so these tests FORCE it -- the paper's own step h = 0.1
 and h = 0.4 -- compare with the oracle at the north_star tolerances, and use the `coarse_steps`
diagnostic output (include/geo.h) to prove how many steps took it; one test straddles |d| = 2^-7 itself.
"""
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


def _run(G, metric, a, st, h, nsteps, host=False, **kw):
    import torch
    ctx = G.geo_create(metric, 1.0, a)
    try:
        n = st.shape[1]
        if host:
            out = G.alloc_outputs_host(n, want_coarse=True)
            G.geo_integrate_host(ctx, np.ascontiguousarray(st), h, nsteps, out, **kw)
            return G.to_numpy(out)
        dev = torch.device("cuda:0")
        out = G.alloc_outputs(n, dev, want_coarse=True)
        G.geo_integrate(ctx, torch.from_numpy(np.ascontiguousarray(st)).to(dev), h, nsteps, out, **kw)
        torch.cuda.synchronize()
        return G.to_numpy(out)
    finally:
        G.geo_destroy(ctx)


@pytest.mark.parametrize("h,nsteps,min_frac", [(0.4, 2500, 0.10), (0.1, 10000, 0.0)])
def test_bound_orbits_coarse_step_vs_oracle(G, oracle, h, nsteps, min_frac):
    """Kerr a = 0.9 bound orbits (the config-2 distribution) to tau = 1000 at the paper's h = 0.1 and at h = 0.4:
    1e-9 against the oracle while a counted share of the steps goes through rk4_sum_full."""
    a = 0.9
    st = W.kerr_bound(3000, a, W.SEED_BASE + 2)
    o = oracle.integrate(oracle.KERR, 1.0, a, st, h, nsteps, nthreads=NCPU)
    g = _run(G, G.KERR, a, st, h, nsteps)
    c = parity.compare(g, o)
    frac = g["coarse_steps"].sum() / float(g["steps_done"].sum())
    print(f"h = {h}: {frac:.4f} of all steps took the full-sin/cos path ({(g['coarse_steps'] > 0).mean():.3f} of the particles "
          f"at least once); max err {c['err'].max():.3e}")
    # reading P3: at h = 0.4 a handful of low-|L_z| orbits blow up (health |2H+1| ~ 1e6, reading B7) and no two FP64
    # evaluations agree on them; every particle the oracle determines to 1e-10 (double vs long double) must be at 1e-9
    def certify(jj):
        sub = np.ascontiguousarray(st[:, jj])
        return [oracle.integrate(oracle.KERR, 1.0, a, sub, h, nsteps, long_double=True, nthreads=NCPU),
                oracle.integrate(oracle.KERR, 1.0, a, parity.ulp_nudged(sub), h, nsteps, nthreads=NCPU)]
    rep = parity.p3_report(g, o, certify, 1e-9, labels=st[[0, 1, 3, 4, 5]], max_fail_frac=0.01, what=f"bound orbits h={h}")
    print(rep)
    assert rep["class_mismatch"] == 0
    assert frac > min_frac and g["coarse_steps"].sum() > 0
    gh = _run(G, G.KERR, a, st[:, :777], h, nsteps, host=True)             # the counter through the host entry point
    assert np.array_equal(gh["coarse_steps"], g["coarse_steps"][:777])


@pytest.mark.parametrize("h", [0.1, 0.4])
def test_near_horizon_rays_coarse_step_vs_oracle(G, oracle, h):
    """Camera rays of config 3 traced with a coarse step: captured rays approach the horizon where every stage angle is
    large.  Class identical and 1e-8 on certified rays (reading P3), fallback share reported."""
    a = 0.998
    full, consts = W.camera_rays(1024, a, 60.0, return_constants=True)
    ii = np.arange(1024 * 1024).reshape(1024, 1024)[300:724:9, 300:724:9].ravel()      # 48 x 48 around the shadow
    st = np.ascontiguousarray(full[:, ii])
    kw = dict(r_capture=W.horizon_radius(1.0, a) + 0.01, r_escape=1100.0)
    ncap = int(round(4000 / h)) * 2
    o = oracle.integrate(oracle.KERR, 1.0, a, st, h, ncap, kind=oracle.NULL, nthreads=NCPU, **kw)
    g = _run(G, G.KERR, a, st, h, ncap, kind=G.NULL, **kw)
    def certify(jj):
        sub = np.ascontiguousarray(st[:, jj])
        okw = dict(kind=oracle.NULL, nthreads=NCPU, **kw)
        return [oracle.integrate(oracle.KERR, 1.0, a, sub, h, ncap, long_double=True, **okw),
                oracle.integrate(oracle.KERR, 1.0, a, parity.ulp_nudged(sub), h, ncap, **okw)]
    rep = parity.p3_report(g, o, certify, 1e-8, labels=consts[:, ii], max_fail_frac=0.05, what=f"near-horizon rays h={h}")
    captured = g["status"] == G.ST_CAPTURED
    print(rep, "fallback steps per captured ray:", g["coarse_steps"][captured].mean(), "per escaped ray:", g["coarse_steps"][~captured].mean())
    assert captured.sum() > 200 and (g["coarse_steps"][captured] > 0).mean() > 0.9


def test_threshold_straddle_single_step(G, oracle):
    """ONE RK4 step of particles that differ only in p_theta, chosen so that the largest stage angle of the step (the
    fourth stage point sits at h * dtheta/dtau) runs from 0.8 x 2^-7 to 1.2 x 2^-7: below the threshold the
    angle-addition kernels are used, above it the full sin/cos path -- the counter must switch exactly once, inside the
    scanned range, and both sides of the switch must agree with the oracle to rounding (1e-14): there is no
    discontinuity between the two evaluations."""
    a, h = 0.9, 0.1
    r0, th0 = 8.0, 1.0
    rho2 = r0 * r0 + a * a * math.cos(th0) ** 2
    n = 513
    d = np.linspace(0.8, 1.2, n) * 2.0 ** -7
    st = np.zeros((6, n))
    st[0], st[1], st[5] = r0, th0, 2.5
    st[4] = d * rho2 / h                                  # h * dtheta/dtau = h p_theta / rho^2 at the base point
    o = oracle.integrate(oracle.KERR, 1.0, a, st, h, 1)
    g = _run(G, G.KERR, a, st, h, 1)
    cs = g["coarse_steps"]
    assert set(np.unique(cs)) == {0, 1} and cs[0] == 0 and cs[-1] == 1
    assert (np.diff(cs) >= 0).all()                       # switches once, monotonically in |d|
    k = int(np.argmax(cs))
    print(f"switch between base-point h*dtheta/dtau = {d[k - 1] * 128:.6f} and {d[k] * 128:.6f} x 2^-7 (particle {k} of {n})")
    assert 8 < k < n - 8
    c = parity.compare(g, o)
    assert c["same_class"].all() and c["err"].max() <= 1e-14, c["err"].max()
