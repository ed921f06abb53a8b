"""Pins of the oracle's adaptive Runge-Kutta 5(4) path (oracle/geo_oracle.cpp).

The paper only announces "others method of the RK family", so there are no printed values:
the pins are the mathematics -- the order conditions of the tableau (Butcher's rooted-tree conditions up to
order 5 for the propagated solution, up to order 4 and NOT 5 for the embedded one), fifth-order convergence
with the controller switched off, agreement with the pinned fixed-step RK4 path at a small step, the
constants of motion, and the analytic capture/escape criterion for camera rays.
"""
import os
import sys

import numpy as np

from paper_1803_08320_b200 import workloads as W

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from test_oracle_integration import _null_class_analytic  # noqa: E402


def test_tableau_order_conditions(oracle):
    T = oracle.dp45_tableau()
    A, c, b5, b4 = T["a"], T["c"], T["b5"], T["b4"]
    assert np.allclose(A.sum(axis=1), c, atol=1e-15)                 # row-sum condition
    assert np.allclose(A[6, :], b5, atol=0) and np.all(np.triu(A) == 0)   # FSAL: last row = weights; explicit
    Ac = A @ c

    def conds(b):
        return {
            1: [(b.sum(), 1.0)],
            2: [(b @ c, 1 / 2)],
            3: [(b @ c**2, 1 / 3), (b @ Ac, 1 / 6)],
            4: [(b @ c**3, 1 / 4), (b @ (c * Ac), 1 / 8), (b @ (A @ c**2), 1 / 12), (b @ (A @ Ac), 1 / 24)],
            5: [(b @ c**4, 1 / 5), (b @ (c**2 * Ac), 1 / 10), (b @ (c * (A @ c**2)), 1 / 15),
                (b @ (c * (A @ Ac)), 1 / 30), (b @ Ac**2, 1 / 20), (b @ (A @ c**3), 1 / 20),
                (b @ (A @ (c * Ac)), 1 / 40), (b @ (A @ (A @ c**2)), 1 / 60), (b @ (A @ (A @ Ac)), 1 / 120)],
        }
    for order, lst in conds(b5).items():
        for got, want in lst:
            assert abs(got - want) < 2e-16 * 8, (order, got, want)
    c4 = conds(b4)
    for order in (1, 2, 3, 4):
        for got, want in c4[order]:
            assert abs(got - want) < 2e-16 * 8, (order, got, want)
    assert max(abs(g - w) for g, w in c4[5]) > 1e-4                  # the embedded solution is 4th order only


def test_fifth_order_convergence_with_fixed_step(oracle):
    a = 0.5
    st = W.kerr_bound(4000, a, W.SEED_BASE + 4)
    st = np.ascontiguousarray(st[:, np.argsort(st[0])[:10]])
    sols = []
    for k in (1, 2, 4):
        n = 400 * k
        r = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.1 / k, np.inf, 1.0, n, long_double=True)
        assert (r["steps_done"] == n).all() and (r["rejected"] == 0).all()
        sols.append(r["final_state"])
    Q = np.linalg.norm(sols[0] - sols[1], axis=0) / np.linalg.norm(sols[1] - sols[2], axis=0)
    assert Q.min() > 20.0 and Q.max() < 60.0 and abs(np.median(Q) - 32.0) < 3.0, Q   # 2^5; RK4 gives 16


def test_adaptive_agrees_with_fixed_step_rk4_at_a_final_time(oracle):
    """The paper's first stop condition, "the final evolution time is reached": both paths
    integrate the same geodesics to the same tau -- bound Kerr orbits to tau = 40 and camera rays to
    tau = 1015 (past the hole) -- and must agree to the tolerance of the coarser one (RK4 at a small h)."""
    a = 0.9
    st = W.kerr_bound(48, a, W.SEED_BASE + 2)
    fx = oracle.integrate(oracle.KERR, 1.0, a, st, 0.0025, 16000, nthreads=8)
    ad = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.01, 1e-13, 1e-13, 100000, tau_end=40.0, nthreads=8)
    assert (ad["status"] == oracle.ST_MAXSTEPS).all() and ad["steps_done"].max() < 4000
    d = np.abs(ad["final_state"] - fx["final_state"]) / np.maximum(np.abs(fx["final_state"]), 1.0)
    assert d.max() < 2e-9, d.max()
    a = 0.998
    full = W.camera_rays(64, a, 60.0)
    ii = np.arange(64 * 64).reshape(64, 64)[3::7, 2::7].ravel()
    st = np.ascontiguousarray(full[:, ii])
    rc = W.horizon_radius(1.0, a) + 0.01
    kw = dict(r_capture=rc, r_escape=1100.0, kind=oracle.NULL, nthreads=8)
    fx = oracle.integrate(oracle.KERR, 1.0, a, st, 0.005, 203000, **kw)
    ad = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.02, 1e-12, 1e-12, 100000, tau_end=1015.0, **kw)
    assert np.array_equal(fx["status"] == oracle.ST_CAPTURED, ad["status"] == oracle.ST_CAPTURED)
    alive = fx["status"] == oracle.ST_MAXSTEPS
    assert alive.sum() > 40 and ad["steps_done"][alive].max() < 3000      # vs 203 000 fixed steps
    d = np.abs(ad["final_state"][:, alive] - fx["final_state"][:, alive]) / np.maximum(np.abs(fx["final_state"][:, alive]), 1.0)
    assert d.max() < 1e-7, d.max()
    assert ad["health"][alive].max() < 1e-9


def test_adaptive_classes_match_the_analytic_criterion(oracle):
    a = 0.998
    st, (al, be, Lz, Q) = W.camera_rays(14, a, 60.0, return_constants=True)
    rp = W.horizon_radius(1.0, a)
    r = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.02, 1e-10, 1e-10, 100000, r_capture=rp + 0.01,
                                  r_escape=1100.0, kind=oracle.NULL, nthreads=8)
    esc = _null_class_analytic(a, Lz, Q, rp, 1000.0)
    assert np.all(np.isin(r["status"], (oracle.ST_CAPTURED, oracle.ST_ESCAPED)))
    assert np.array_equal(r["status"] == oracle.ST_ESCAPED, esc)
    assert np.abs(r["final_state"][4] - 1.0).max() < 1e-12 and np.array_equal(r["final_state"][7], st[5])


def test_adaptive_bound_orbits_conserve_the_constants(oracle):
    a = 0.9
    st, (E, Lz, Q) = W.kerr_bound(64, a, W.SEED_BASE + 2, return_constants=True)
    r = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.01, 1e-12, 1e-12, 4000)
    f = r["final_state"]
    assert (r["status"] == oracle.ST_MAXSTEPS).all() and (r["steps_done"] + r["rejected"] == 4000).all()
    assert r["health"].max() < 1e-9
    Qf = f[6] ** 2 + np.cos(f[2]) ** 2 * (a * a * (1 - f[4] ** 2) + f[7] ** 2 / np.sin(f[2]) ** 2)
    assert np.abs(Qf - Q).max() < 1e-8 and f[0].min() > 100.0      # far fewer steps than h = 0.01 would need


def test_undefined_error_estimate_shrinks_the_step_and_ends_with_numeric(oracle):
    """Reading A2 (round 2): radial infall in Schwarzschild with L = 0 keeps phi exactly 0, so with atol = 0 the scaled
    error of phi is 0/0 on every attempt.  The attempt is rejected with factor 0.2 until the step falls below h_min
    (NUMERIC) -- it must not be retried unchanged until max_attempts.  With h_min = 0 the step shrinks to exactly zero
    and the particle ends the same way."""
    st = np.array([[8.0], [np.pi / 2], [0.0], [-0.1], [0.0], [0.0]])
    r = oracle.integrate_adaptive(oracle.SCHWARZSCHILD, 1.0, 0.0, st, 0.1, 1e-9, 0.0, 10**6, h_min=1e-12)
    assert r["status"][0] == oracle.ST_NUMERIC and r["steps_done"][0] == 0
    assert r["rejected"][0] == 16               # 0.1 * 0.2^16 = 6.6e-13 < 1e-12 <= 0.1 * 0.2^15
    r0 = oracle.integrate_adaptive(oracle.SCHWARZSCHILD, 1.0, 0.0, st, 0.1, 1e-9, 0.0, 10**6, h_min=0.0)
    assert r0["status"][0] == oracle.ST_NUMERIC and 400 < r0["rejected"][0] < 500      # 0.2^k underflows to 0 near k = 463
    np.testing.assert_array_equal(r0["final_state"][1:4, 0], st[0:3, 0])               # final = y0, untouched


# ---- reading A3: dense output of the pair (records at fixed tau from the continuous extension) ----------------------
def _tree_sums(T, w):
    A, c = T["a"], T["c"]
    Ac = A @ c
    return [(w.sum(), 1, 1.0), (w @ c, 2, 2.0), (w @ c**2, 3, 3.0), (w @ Ac, 3, 6.0), (w @ c**3, 4, 4.0), (w @ (c * Ac), 4, 8.0),
            (w @ (A @ c**2), 4, 12.0), (w @ (A @ Ac), 4, 24.0)]


def test_dense_output_weights_are_a_fourth_order_hermite_extension(oracle):
    """w_i(theta) of reading A3 against what defines a continuous extension of order 4 (Hairer, Norsett & Wanner II.6):
    the order conditions sum_i w_i(theta) Phi_i(tree) = theta^q / gamma(tree) for all 8 rooted trees with q <= 4, at
    several theta -- a wrong coefficient d_i, a swapped stage or a wrong power of theta violates one of them -- and the
    Hermite end conditions w(0) = 0, w(1) = b (the 5th-order weights), w'(0) = e_1, w'(1) = e_7 (C^1 across steps)."""
    T = oracle.dp45_tableau()
    for th in (0.0, 0.1, 1.0 / 3.0, 0.5, 0.77, 1.0):
        w = oracle.dp45_dense_weights(th)
        for got, q, gamma in _tree_sums(T, w):
            assert abs(got - th**q / gamma) < 4e-16, (th, q, gamma, got)
    assert np.all(oracle.dp45_dense_weights(0.0) == 0.0)
    assert np.allclose(oracle.dp45_dense_weights(1.0), T["b5"], rtol=0, atol=1e-16)
    e = 1e-6
    d0 = (oracle.dp45_dense_weights(e) - oracle.dp45_dense_weights(0.0)) / e
    d1 = (oracle.dp45_dense_weights(1.0) - oracle.dp45_dense_weights(1.0 - e)) / e
    assert np.allclose(d0, np.eye(7)[0], atol=1e-5) and np.allclose(d1, np.eye(7)[6], atol=1e-5)
    # it is NOT fifth order (the extension is one order below the propagated solution): the q = 5 bushy tree fails
    w = oracle.dp45_dense_weights(0.5)
    assert abs(w @ T["c"]**4 - 0.5**5 / 5.0) > 1e-6


def test_dense_output_records_converge_with_fourth_order_and_match_step_states(oracle):
    a = 0.5
    st = W.kerr_bound(4000, a, W.SEED_BASE + 4)
    st = np.ascontiguousarray(st[:, np.argsort(st[0])[:8]])
    T_end, dtau = 24.0, 0.7                       # record times are NOT multiples of the step
    ncap = int(T_end / dtau) + 2
    ref = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.0125, np.inf, 1.0, 10**6, tau_end=T_end, snap_dtau=dtau,
                                    snap_capacity=ncap, long_double=True)
    errs = []
    for k in (1, 2, 4):
        r = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.4 / k, np.inf, 1.0, 10**6, tau_end=T_end, snap_dtau=dtau,
                                      snap_capacity=ncap, long_double=True)
        assert (r["snap_count"] == 1 + int(T_end / dtau)).all() and (r["rejected"] == 0).all()
        valid = r["snapshots"][:, : 1 + int(T_end / dtau), :]
        errs.append(np.abs(valid - ref["snapshots"][:, : 1 + int(T_end / dtau), :]).max(axis=(1, 2)))
        assert np.isnan(r["snapshots"][:, 1 + int(T_end / dtau):, :]).all()          # nothing beyond the final time
    q1, q2 = errs[0] / errs[1], errs[1] / errs[2]
    assert np.median(q1) > 12.0 and np.median(q2) > 12.0, (q1, q2)                   # >= 2^4 up to the 5th-order part
    assert errs[2].max() < 1e-6
    # slot 0 = y0; a record that falls on a step boundary is that step's state (theta = 1: w = b)
    h, every = 0.25, 4                                                                # records at tau = 1, 2, ...
    r = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, h, np.inf, 1.0, 10**6, tau_end=6.0, snap_dtau=h * every, snap_capacity=8)
    assert (r["snap_count"] == 7).all()
    assert np.array_equal(r["snapshots"][:, 0, [1, 2, 3, 5, 6, 7]], st.T) and (r["snapshots"][:, 0, 0] == 0).all()
    for j in (1, 3, 6):
        rj = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, h, np.inf, 1.0, 10**6, tau_end=j * h * every)
        assert np.abs(r["snapshots"][:, j, :] - rj["final_state"].T).max() < 1e-13


def test_dense_output_stops_with_the_ray_and_respects_capacity(oracle):
    a = 0.998
    st = np.ascontiguousarray(W.camera_rays(64, a, 60.0)[:, ::37])
    rc = W.horizon_radius(1.0, a) + 0.01
    r = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.02, 1e-9, 1e-9, 200000, r_capture=rc, r_escape=1100.0,
                                  kind=oracle.NULL, snap_dtau=25.0, snap_capacity=40, snap_mask=0x0F)
    tau_rec = (r["snap_count"] - 1) * 25.0                        # time of the last record of each ray
    t_last = r["final_state"][0]
    assert (r["snap_count"] >= 40).all()                          # ~2100 M of affine time: capacity 40 overflows (S3) ...
    assert np.isfinite(r["snapshots"]).all()                      # ... all 40 slots written, none beyond
    full = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.02, 1e-9, 1e-9, 200000, r_capture=rc, r_escape=1100.0,
                                     kind=oracle.NULL, snap_dtau=25.0, snap_capacity=200, snap_mask=0x0F)
    assert np.array_equal(full["snap_count"], r["snap_count"]) and np.array_equal(full["snapshots"][:, :40], r["snapshots"])
    cnt = full["snap_count"]
    for i in range(st.shape[1]):
        assert np.isnan(full["snapshots"][i, cnt[i]:]).all() and np.isfinite(full["snapshots"][i, : cnt[i]]).all()
        tt = full["snapshots"][i, : cnt[i], 0]
        assert (np.diff(tt) > 0).all() and tt[-1] <= t_last[i] + 1e-9            # coordinate time increases along the ray
    assert (tau_rec > 0).all()
