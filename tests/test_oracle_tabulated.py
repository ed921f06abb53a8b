"""Pins of the tabulated-metric oracle (oracle/geo_tab_oracle.cpp, readings T1-T5).

The paper only announces numerical metrics, so nothing is printed: the pins are the
mathematics.  Interpolant: Keys' cubic-convolution KERNEL form summed over all nodes (the oracle uses the four
per-cell weight polynomials), node values, exactness on quadratics, C^1 continuity.  Equations of motion: finite
differences of H on a metric whose fields are quadratic polynomials (there the interpolant IS the metric, so a
dropped term, a wrong sign or swapped derivatives in the RHS fail).  Integration: flat space in spherical
coordinates against the straight line's closed form; the Kerr metric of eq.(8) sampled on a grid against the pinned
analytic-metric oracle, with the convergence order in the grid spacing; constants of motion; stop rules.
"""
import math

import numpy as np

from paper_1803_08320_b200 import workloads as W


def _rand_table(n1=12, n2=10, seed=1):
    rng = np.random.default_rng(seed)
    return {"tab": np.ascontiguousarray(rng.uniform(0.5, 2.0, (5, n2, n1))), "x1_0": 2.0, "d1": 0.25, "x2_0": -0.3, "d2": 0.4}


def _keys_kernel(s):
    """Keys (1981) eq.(15): u(s) for a = -1/2."""
    s = np.abs(s)
    return np.where(s < 1, 1.5 * s**3 - 2.5 * s**2 + 1, np.where(s < 2, -0.5 * s**3 + 2.5 * s**2 - 4 * s + 2, 0.0))


def _keys_kernel_prime(s):
    sg, s = np.sign(s), np.abs(s)
    return sg * np.where(s < 1, 4.5 * s**2 - 5 * s, np.where(s < 2, -1.5 * s**2 + 5 * s - 4, 0.0))


def test_interpolant_equals_the_kernel_form_summed_over_all_nodes(tab_oracle):
    tb = _rand_table()
    n2, n1 = tb["tab"].shape[1:]
    xs1 = tb["x1_0"] + tb["d1"] * np.arange(n1)
    xs2 = tb["x2_0"] + tb["d2"] * np.arange(n2)
    rng = np.random.default_rng(2)
    for _ in range(200):
        x1 = rng.uniform(xs1[1], xs1[n1 - 2] - 1e-9)
        x2 = rng.uniform(xs2[1], xs2[n2 - 2] - 1e-9)
        k1, k2 = _keys_kernel((x1 - xs1) / tb["d1"]), _keys_kernel((x2 - xs2) / tb["d2"])
        d1, d2 = _keys_kernel_prime((x1 - xs1) / tb["d1"]) / tb["d1"], _keys_kernel_prime((x2 - xs2) / tb["d2"]) / tb["d2"]
        v, g1, g2 = tab_oracle.fields(tb, x1, x2)
        for f in range(5):
            T = tb["tab"][f]
            assert abs(v[f] - k2 @ T @ k1) < 1e-13
            assert abs(g1[f] - k2 @ T @ d1) < 1e-12
            assert abs(g2[f] - d2 @ T @ k1) < 1e-12


def test_interpolant_passes_through_the_nodes_and_domain_is_where_the_stencil_exists(tab_oracle):
    tb = _rand_table()
    n2, n1 = tb["tab"].shape[1:]
    for j in range(n2):
        for i in range(n1):
            r = tab_oracle.fields(tb, tb["x1_0"] + tb["d1"] * i, tb["x2_0"] + tb["d2"] * j)
            inside = 1 <= i <= n1 - 3 and 1 <= j <= n2 - 3              # reading T4
            assert (r is not None) == inside, (i, j)
            if inside:
                assert np.allclose(r[0], tb["tab"][:, j, i], rtol=0, atol=1e-14)
    assert tab_oracle.fields(tb, float("nan"), 0.5) is None


def test_interpolant_is_exact_on_quadratics_and_C1_across_cells(tab_oracle):
    n1, n2 = 14, 11
    tb = {"x1_0": 1.0, "d1": 0.5, "x2_0": 0.2, "d2": 0.3}
    X1, X2 = np.meshgrid(tb["x1_0"] + tb["d1"] * np.arange(n1), tb["x2_0"] + tb["d2"] * np.arange(n2))
    c = np.random.default_rng(3).uniform(-1, 1, (5, 3, 3))

    def poly(f, x1, x2, d1=0, d2=0):
        p1 = [np.ones_like(x1), x1, x1 * x1] if d1 == 0 else [0 * x1, np.ones_like(x1), 2 * x1]
        p2 = [np.ones_like(x2), x2, x2 * x2] if d2 == 0 else [0 * x2, np.ones_like(x2), 2 * x2]
        return sum(c[f, i, j] * p1[i] * p2[j] for i in range(3) for j in range(3))
    tb["tab"] = np.ascontiguousarray(np.stack([poly(f, X1, X2) for f in range(5)]))
    rng = np.random.default_rng(4)
    for _ in range(100):
        x1, x2 = np.float64(rng.uniform(1.6, 6.9)), np.float64(rng.uniform(0.55, 2.8))
        v, g1, g2 = tab_oracle.fields(tb, x1, x2)
        for f in range(5):
            assert abs(v[f] - poly(f, x1, x2)) < 2e-12
            assert abs(g1[f] - poly(f, x1, x2, d1=1)) < 2e-11
            assert abs(g2[f] - poly(f, x1, x2, d2=1)) < 2e-11
    # C^1 across a cell face on a NON-polynomial table
    tr = _rand_table()
    xb = tr["x1_0"] + 4 * tr["d1"]
    lo, hi = tab_oracle.fields(tr, xb - 1e-10, 0.77), tab_oracle.fields(tr, xb + 1e-10, 0.77)
    for k in range(3):
        assert np.max(np.abs(lo[k] - hi[k])) < 1e-7
    yb = tr["x2_0"] + 5 * tr["d2"]
    lo, hi = tab_oracle.fields(tr, 3.21, yb - 1e-10), tab_oracle.fields(tr, 3.21, yb + 1e-10)
    for k in range(3):
        assert np.max(np.abs(lo[k] - hi[k])) < 1e-7


def _quadratic_metric():
    """A made-up stationary axisymmetric metric whose five fields are quadratics: the interpolant is exact on it."""
    def fields(x1, x2):
        return (1.0 + 0.05 * x1 + 0.02 * x2 * x2 - 0.01 * x1 * x2,          # alpha
                -0.03 + 0.004 * x1 * x1 - 0.01 * x2,                        # beta^phi
                1.5 + 0.1 * x1 * x1 + 0.05 * x2,                            # gamma_11
                2.0 + 0.3 * x1 + 0.2 * x2 * x2,                             # gamma_22
                1.0 + 0.5 * x1 * x2 + 0.1 * x1 * x1)                        # gamma_33
    n1, n2 = 20, 18
    tb = {"x1_0": 0.5, "d1": 0.2, "x2_0": 0.4, "d2": 0.15}
    X1, X2 = np.meshgrid(tb["x1_0"] + tb["d1"] * np.arange(n1), tb["x2_0"] + tb["d2"] * np.arange(n2))
    tb["tab"] = np.ascontiguousarray(np.stack(fields(X1, X2)))
    return tb, fields


def test_rhs_is_hamiltons_equations_of_the_3p1_hamiltonian(tab_oracle):
    """eqs.(3),(4) PAPER.md:60-65: dx/dtau = dH/dp, dp/dtau = -dH/dx with H = 1/2 g^{mu nu} p_mu p_nu built
    here by inverting the 4x4 matrix of line element (1) -- not from the 3+1 closed form."""
    tb, fields = _quadratic_metric()

    def H(x1, x2, pt, p1, p2, pph):
        al, be, g11, g22, g33 = fields(x1, x2)
        g = np.zeros((4, 4))                       # t, x1, x2, phi
        g[0, 0] = -al * al + g33 * be * be
        g[0, 3] = g[3, 0] = g33 * be
        g[1, 1], g[2, 2], g[3, 3] = g11, g22, g33
        p = np.array([pt, p1, p2, pph])
        return 0.5 * p @ np.linalg.inv(g) @ p
    rng = np.random.default_rng(5)
    for _ in range(50):
        x1, x2 = rng.uniform(1.0, 3.8), rng.uniform(0.7, 2.6)
        E, p1, p2, L = rng.uniform(0.5, 2), rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-2, 2)
        d, Hval = tab_oracle.rhs(tb, [0.0, x1, x2, 0.0, E, p1, p2, L])
        args = np.array([x1, x2, -E, p1, p2, L])
        e = 1e-5

        def dH(k):
            up, dn = args.copy(), args.copy()
            up[k] += e
            dn[k] -= e
            return (H(*up) - H(*dn)) / (2 * e)
        want = np.array([dH(2), dH(3), dH(4), dH(5), -dH(0), -dH(1)])       # t, x1, x2, phi, p1, p2
        assert abs(Hval - H(*args)) < 1e-13
        assert np.max(np.abs(d - want)) < 2e-9, (d, want)


def _flat_table(n1, n2, r_lo=0.5, r_hi=12.0):
    d1, d2 = (r_hi - r_lo) / (n1 - 1), math.pi / (n2 - 1)            # n2 odd => theta = pi/2 is a node
    x1 = r_lo + d1 * (np.arange(n1 + 4) - 2)
    x2 = d2 * (np.arange(n2 + 4) - 2)
    R, TH = np.meshgrid(x1, x2)
    tab = np.stack([np.ones_like(R), np.zeros_like(R), np.ones_like(R), R * R, R * R * np.sin(TH) ** 2])
    return {"tab": np.ascontiguousarray(tab), "x1_0": float(x1[0]), "d1": d1, "x2_0": float(x2[0]), "d2": d2}


def test_flat_space_geodesics_are_straight_lines(tab_oracle):
    """Minkowski space in spherical coordinates (alpha = 1, beta = 0, gamma = diag(1, r^2, r^2 sin^2 theta)): in the
    plane theta = pi/2 (a grid line, where the interpolated sin^2 is exactly 1 with zero theta-derivative by symmetry
    and r^2 is a quadratic) the tabulated metric is exact, so RK4 must follow x(tau) = x0 + u tau, t = sqrt(1+u^2) tau."""
    tb = _flat_table(47, 33)
    x0, u = np.array([3.0, -2.0]), np.array([-0.3, 0.8])
    r0 = np.hypot(*x0)
    st = np.array([[r0], [math.pi / 2], [math.atan2(x0[1], x0[0])], [x0 @ u / r0], [0.0], [x0[0] * u[1] - x0[1] * u[0]]])
    errs = []
    for h, n in ((0.02, 400), (0.01, 800)):
        o = tab_oracle.integrate(tb, st, h, n)
        assert o["status"][0] == tab_oracle.ST_MAXSTEPS and o["steps_done"][0] == n
        xe = x0 + u * h * n
        t, r, th, ph, E = o["final_state"][:5, 0]
        assert abs(th - math.pi / 2) < 1e-13                 # symmetric stencil: zero theta-force up to rounding
        assert abs(E - math.sqrt(1 + u @ u)) < 1e-15
        errs.append(max(abs(r - np.hypot(*xe)), abs(ph - math.atan2(xe[1], xe[0])), abs(t - E * h * n)))
    assert errs[0] < 1e-7 and 10 < errs[0] / errs[1] < 22, errs          # fourth order in h, nothing else
    # off the plane sin^2 is only interpolated: the error falls with the grid spacing (reading T2: the force is
    # second-order accurate)
    x0, u = np.array([3.0, -2.0, 1.0]), np.array([-0.3, 0.8, 0.2])
    r0 = np.linalg.norm(x0)
    th0, ph0 = math.acos(x0[2] / r0), math.atan2(x0[1], x0[0])
    er, et, ep = (np.array([math.sin(th0) * math.cos(ph0), math.sin(th0) * math.sin(ph0), math.cos(th0)]),
                  np.array([math.cos(th0) * math.cos(ph0), math.cos(th0) * math.sin(ph0), -math.sin(th0)]),
                  np.array([-math.sin(ph0), math.cos(ph0), 0.0]))
    st = np.array([[r0], [th0], [ph0], [u @ er], [r0 * (u @ et)], [r0 * math.sin(th0) * (u @ ep)]])
    xe = x0 + u * 4.0
    errs = []
    for n2 in (33, 65, 129):
        o = tab_oracle.integrate(_flat_table(47, n2), st, 0.01, 400)
        r, th, ph = o["final_state"][1:4, 0]
        got = r * np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
        errs.append(np.linalg.norm(got - xe))
    assert errs[2] < 2e-5 and errs[0] / errs[1] > 3 and errs[1] / errs[2] > 3, errs


def test_tabulated_kerr_rhs_converges_to_the_analytic_metric(tab_oracle, oracle):
    """eq.(8) PAPER.md:97 sampled on a grid: the interpolated RHS tends to the analytic-metric oracle's (itself pinned
    in test_oracle_pins.py) -- velocities with the third-order value error, forces with the second-order derivative error."""
    a = 0.9
    rng = np.random.default_rng(6)
    pts = [(rng.uniform(3, 20), rng.uniform(0.6, 2.5), rng.uniform(0.9, 1.0), rng.uniform(-0.3, 0.3), rng.uniform(-2, 2),
            rng.uniform(-3, 3)) for _ in range(400)]
    ev, ef = [], []
    for n1, n2 in ((257, 65), (513, 129), (1025, 257)):
        tb = W.kerr_metric_table(1.0, a, n1, n2, 2.0, 24.0, 0.3, math.pi - 0.3)
        mv = mf = 0.0
        for r, th, E, pr, pth, L in pts:
            y = [0.0, r, th, 0.0, E, pr, pth, L]
            d, Hval = tab_oracle.rhs(tb, y)
            want = oracle.rhs(oracle.KERR, 1.0, a, y)
            mv = max(mv, np.max(np.abs(d[:4] - want[:4]) / np.maximum(np.abs(want[:4]), 1e-2)))
            mf = max(mf, np.max(np.abs(d[4:] - want[4:])))
        ev.append(mv)
        ef.append(mf)
    assert ev[2] < 1e-6 and ef[2] < 1e-4, (ev, ef)
    assert ev[0] / ev[1] > 5 and ev[1] / ev[2] > 5, ev            # ~8 = 2^3
    assert 3 < ef[0] / ef[1] and 3 < ef[1] / ef[2], ef            # ~4 = 2^2


def test_tabulated_kerr_orbits_converge_to_the_analytic_oracle_in_both_radial_coordinates(tab_oracle, oracle):
    a = 0.9
    st = W.kerr_bound(48, a, W.SEED_BASE + 2)
    ref = oracle.integrate(oracle.KERR, 1.0, a, st, 0.01, 1500)
    rp = W.horizon_radius(1.0, a)
    for radial, lo, hi in (("r", 1.8, 40.0), ("log", math.log(1.8 - rp), math.log(40.0 - rp))):
        errs = []
        for n1, n2 in ((513, 129), (2049, 513)):
            tb = W.kerr_metric_table(1.0, a, n1, n2, lo, hi, 0.2, math.pi - 0.2, radial=radial)
            s = W.to_log_radial(st, rp) if radial == "log" else st
            o = tab_oracle.integrate(tb, s, 0.01, 1500)
            assert (o["status"] == tab_oracle.ST_MAXSTEPS).all()
            f = o["final_state"].copy()
            if radial == "log":                                   # back to Boyer-Lindquist r, p_r
                f[5] = f[5] / np.exp(f[1])
                f[1] = rp + np.exp(f[1])
            assert np.array_equal(f[7], st[5])                    # p_phi is a constant of motion exactly
            # E is derived from the interpolated metric at y0 and then constant
            assert np.max(np.abs(f[4] - ref["final_state"][4])) < 1e-6
            assert np.nanmax(o["health"]) < 1e-7                  # 2H + 1 drift: RK4 + the C^1 interpolant
            errs.append(np.max(np.abs(f[[0, 1, 2, 3, 5, 6]] - ref["final_state"][[0, 1, 2, 3, 5, 6]])
                               / np.maximum(np.abs(ref["final_state"][[0, 1, 2, 3, 5, 6]]), 1.0)))
            if radial == "r" and n1 == 2049:
                # equatorial-crossing event (B5): same particles cross, at the analytic oracle's radius
                crossed = ~np.isnan(ref["eq_cross_r"])
                assert crossed.sum() > 5 and np.array_equal(~np.isnan(o["eq_cross_r"]), crossed)
                assert np.max(np.abs(o["eq_cross_r"][crossed] - ref["eq_cross_r"][crossed])) < 1e-5
        assert errs[1] < 2e-5 and errs[0] / errs[1] > 6, (radial, errs)


def test_stop_rules_and_domain_exit(tab_oracle, oracle):
    a = 0.998
    rp = W.horizon_radius(1.0, a)
    tb = W.kerr_metric_table(1.0, a, 769, 257, math.log(0.005), math.log(60.0), 0.0, math.pi, radial="log", ghost=3)
    full = W.camera_rays(64, a, 60.0, r_obs=50.0)
    ii = np.arange(64 * 64).reshape(64, 64)[4::8, 2::8].ravel()
    st = np.ascontiguousarray(full[:, ii])
    s = W.to_log_radial(st, rp)
    xc, xe = math.log(0.01), math.log(55.0 - rp)
    o = tab_oracle.integrate(tb, s, 0.02, 20000, r_capture=xc, r_escape=xe, kind=tab_oracle.NULL)
    ref = oracle.integrate(oracle.KERR, 1.0, a, st, 0.02, 20000, r_capture=rp + 0.01, r_escape=55.0, kind=oracle.NULL)
    assert set(np.unique(o["status"])) == {tab_oracle.ST_CAPTURED, tab_oracle.ST_ESCAPED}
    assert (o["status"] == ref["status"]).mean() >= 0.97          # same image up to rays grazing the critical curve
    esc = o["status"] == tab_oracle.ST_ESCAPED
    assert (o["final_state"][1][esc] > xe).all() and (o["final_state"][1][~esc] >= xc).all()
    # B1 / T4 on y0, B4, and leaving the table
    y0 = np.array([[1.0, -9.0, 1.0, 1.0, 1.0], [1.5, 1.5, 1.5, 1.5, -0.5], [0.0] * 5, [0.0] * 5, [0.0] * 5, [2.0] * 5])
    y0[1, 2] = float("nan")             # (a NaN x^1 fails the NaN-safe capture test first: B1)
    y0[0, 3] = 4.5                      # beyond the last interior node (x1 <= ln 60 + ghosts)
    o = tab_oracle.integrate(tb, y0, 0.02, 0, r_capture=-6.0, r_escape=9.0)
    assert o["status"].tolist() == [tab_oracle.ST_MAXSTEPS, tab_oracle.ST_CAPTURED, tab_oracle.ST_NUMERIC,
                                    tab_oracle.ST_OUTSIDE, tab_oracle.ST_OUTSIDE]
    assert (o["steps_done"] == 0).all() and np.isnan(o["health"][3])
    # an outgoing timelike particle with no escape radius runs off the table: OUTSIDE, last state inside the domain
    out = np.array([[math.log(30.0)], [1.2], [0.0], [40.0], [0.0], [1.0]])
    o = tab_oracle.integrate(tb, out, 0.05, 100000)
    hi = tb["x1_0"] + tb["d1"] * (tb["tab"].shape[2] - 2)
    assert o["status"][0] == tab_oracle.ST_OUTSIDE and 0 < o["steps_done"][0] < 100000
    assert o["final_state"][1, 0] < hi and o["final_state"][1, 0] > hi - 0.2


# ---- reading T6: GENERAL stationary axisymmetric 3+1 metric (ten fields) ------------------------------------------------
def _quadratic_general_metric():
    """A made-up metric with ALL ten fields non-trivial quadratics (non-zero beta^1, beta^2, off-diagonal gamma_ij),
    gamma_ij positive definite on the grid: the interpolant is exact on it."""
    def fields(x1, x2):
        return (1.0 + 0.05 * x1 + 0.02 * x2 * x2 - 0.01 * x1 * x2,          # alpha
                0.02 + 0.01 * x1 - 0.004 * x2 * x2,                         # beta^1
                -0.015 + 0.006 * x1 * x2,                                   # beta^2
                -0.03 + 0.004 * x1 * x1 - 0.01 * x2,                        # beta^3
                1.5 + 0.1 * x1 * x1 + 0.05 * x2,                            # gamma_11
                0.10 + 0.02 * x1 - 0.03 * x2,                               # gamma_12
                -0.20 + 0.05 * x2 * x2 + 0.01 * x1,                         # gamma_13
                2.0 + 0.3 * x1 + 0.2 * x2 * x2,                             # gamma_22
                0.15 - 0.02 * x1 * x2,                                      # gamma_23
                1.0 + 0.5 * x1 * x2 + 0.1 * x1 * x1)                        # gamma_33
    n1, n2 = 20, 18
    tb = {"x1_0": 0.5, "d1": 0.2, "x2_0": 0.4, "d2": 0.15}
    X1, X2 = np.meshgrid(tb["x1_0"] + tb["d1"] * np.arange(n1), tb["x2_0"] + tb["d2"] * np.arange(n2))
    tb["tab"] = np.ascontiguousarray(np.stack(fields(X1, X2)))
    return tb, fields


def test_general_rhs_is_hamiltons_equations_of_line_element_1(tab_oracle):
    """Reading T6 against eqs.(3),(4) PAPER.md:60-65 with H = 1/2 g^{mu nu} p_mu p_nu built here by inverting the full
    4x4 matrix of line element (1) PAPER.md:47 (g_tt = -alpha^2 + beta_k beta^k, g_ti = gamma_ij beta^j, g_ij = gamma_ij):
    a dropped shift component, a wrong sign, a missing factor 2 on an off-diagonal term or swapped gradients fail it.
    Also the mass-shell energy: H(E) = -kappa/2."""
    tb, fields = _quadratic_general_metric()

    def H(x1, x2, pt, p1, p2, pph):
        al, b1, b2, b3, g11, g12, g13, g22, g23, g33 = fields(x1, x2)
        gam = np.array([[g11, g12, g13], [g12, g22, g23], [g13, g23, g33]])
        bu = np.array([b1, b2, b3])
        bl = gam @ bu
        g = np.zeros((4, 4))                       # t, x1, x2, phi
        g[0, 0] = -al * al + bl @ bu
        g[0, 1:] = g[1:, 0] = bl
        g[1:, 1:] = gam
        p = np.array([pt, p1, p2, pph])
        return 0.5 * p @ np.linalg.inv(g) @ p
    rng = np.random.default_rng(6)
    for _ in range(50):
        x1, x2 = rng.uniform(1.0, 3.8), rng.uniform(0.7, 2.6)
        E, p1, p2, L = rng.uniform(0.5, 2), rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-2, 2)
        kappa = float(rng.integers(0, 2))
        d, Hval, Ems = tab_oracle.rhs_general(tb, [0.0, x1, x2, 0.0, E, p1, p2, L], kappa)
        args = np.array([x1, x2, -E, p1, p2, L])
        e = 1e-5

        def dH(k):
            up, dn = args.copy(), args.copy()
            up[k] += e
            dn[k] -= e
            return (H(*up) - H(*dn)) / (2 * e)
        want = np.array([dH(2), dH(3), dH(4), dH(5), -dH(0), -dH(1)])       # t, x1, x2, phi, p1, p2
        assert abs(Hval - H(*args)) < 1e-13
        assert np.max(np.abs(d - want)) < 2e-9, (d, want)
        assert abs(2.0 * H(x1, x2, -Ems, p1, p2, L) + kappa) < 1e-12        # eq.(5): the energy is ON the mass shell
        assert Ems + (fields(x1, x2)[1] * p1 + fields(x1, x2)[2] * p2 + fields(x1, x2)[3] * L) > 0   # future-directed root


def test_general_layout_reduces_to_the_eq8_structure(tab_oracle):
    """T6 with beta^1 = beta^2 = 0 and a diagonal 3-metric IS T3: the same Kerr table in both layouts gives the same
    right-hand side (1e-14) and the same orbits (1e-12) as the five-field oracle pinned above."""
    a = 0.9
    tb5 = W.kerr_metric_table(1.0, a, 257, 65, 1.8, 40.0, 0.2, math.pi - 0.2)
    tb10 = W.general_table_from_diagonal(tb5)
    st = W.kerr_bound(200, a, W.SEED_BASE + 2)
    for i in range(0, 200, 17):
        y8 = [0.0, st[0, i], st[1, i], 0.0, 0.95, st[3, i], st[4, i], st[5, i]]
        d5, H5 = tab_oracle.rhs(tb5, y8)
        d10, H10, _ = tab_oracle.rhs_general(tb10, y8)
        assert np.max(np.abs(d5 - d10) / np.maximum(np.abs(d5), 1.0)) < 1e-14 and abs(H5 - H10) < 1e-14
    o5 = tab_oracle.integrate(tb5, st, 0.01, 2000)
    o10 = tab_oracle.integrate_general(tb10, st, 0.01, 2000)
    assert np.array_equal(o5["status"], o10["status"]) and np.array_equal(o5["steps_done"], o10["steps_done"])
    assert np.max(np.abs(o5["final_state"] - o10["final_state"]) / np.maximum(np.abs(o5["final_state"]), 1.0)) < 1e-12


def test_kerr_schild_table_reproduces_boyer_lindquist_orbits_and_penetrates_the_horizon(tab_oracle, oracle):
    """The Kerr metric in ingoing Kerr-Schild coordinates (beta^r != 0, gamma_r phi != 0: outside eq.(8)'s structure) through
    the general tabulated path against the pinned ANALYTIC Boyer-Lindquist oracle.  r, theta, p_theta, E, L are the same in
    both coordinate systems (only t and phi are re-labelled), so bound orbits must agree in them, the better the finer
    the grid; and a plunging particle crosses r_+ with finite state and |2H + 1| small -- in Boyer-Lindquist coordinates
    the same particle cannot be followed through (Delta = 0)."""
    a, M = 0.9, 1.0
    st, consts = W.kerr_bound(40, a, W.SEED_BASE + 2, return_constants=True)
    E = consts[0]
    ob = oracle.integrate(oracle.KERR, M, a, st, 0.01, 3000)
    assert np.allclose(ob["final_state"][4], E, rtol=0, atol=1e-12)          # the generator's E is the mass-shell E
    ks = W.to_kerr_schild(st, E, M, a)
    errs = []
    for n1, n2 in ((513, 129), (1025, 257)):
        tb = W.kerr_schild_metric_table(M, a, n1, n2, 1.2, 40.0, 0.15, math.pi - 0.15)
        og = tab_oracle.integrate_general(tb, ks, 0.01, 3000)
        assert (og["status"] == tab_oracle.ST_MAXSTEPS).all()
        assert np.max(np.abs(og["final_state"][4] - E)) < 2e-6 * (513 / n1) ** 2   # E of the interpolated metric's mass shell
        assert np.array_equal(og["final_state"][7], st[5])
        errs.append(np.abs(og["final_state"][[1, 2, 6]] - ob["final_state"][[1, 2, 6]]).max())
    assert errs[1] < errs[0] / 3.0 and errs[1] < 2e-4, errs            # O(d^2) force error of the interpolant: x ~5 per halving
    # horizon penetration: radial-ish infall from r = 6 through r_+ = 1.4359 down to r ~ 1.3 (inside the table)
    rp = M + math.sqrt(M * M - a * a)
    fall = np.array([[6.0], [1.2], [0.0], [0.0], [0.3], [1.0]])               # BL data at rest-ish with L = 1
    Ef = oracle.integrate(oracle.KERR, M, a, fall, 0.01, 0)["final_state"][4]
    kf = W.to_kerr_schild(fall, Ef, M, a)
    tb = W.kerr_schild_metric_table(M, a, 1025, 257, 1.2, 40.0, 0.15, math.pi - 0.15)
    og = tab_oracle.integrate_general(tb, kf, 0.005, 20000, r_capture=1.3)
    assert og["status"][0] == tab_oracle.ST_CAPTURED and og["final_state"][1, 0] < rp - 0.05      # went INSIDE the horizon
    assert np.isfinite(og["final_state"]).all() and og["health"][0] < 1e-5


def test_tabulated_trajectory_records_follow_S1_to_S3(tab_oracle):
    """Records on the tabulated path (round 2): slot 0 = y0 with the mass-shell E, slot j = the state after j *
    snapshot_every accepted steps -- bitwise the final state of a run of that length (SURVEY 8(c) pin 'Snapshots') --,
    nothing after termination, records beyond the capacity dropped but counted, components by mask."""
    a = 0.9
    tb = W.kerr_metric_table(1.0, a, 257, 65, 1.8, 40.0, 0.2, math.pi - 0.2)
    st = W.kerr_bound(60, a, W.SEED_BASE + 2)
    r = tab_oracle.integrate(tb, st, 0.01, 900, snapshot_every=300)
    assert (r["snap_count"] == 4).all() and r["snapshots"].shape == (60, 4, 8)
    assert np.array_equal(r["snapshots"][:, 0, [1, 2, 3, 5, 6, 7]], st.T) and (r["snapshots"][:, 0, 0] == 0).all()
    assert np.array_equal(r["snapshots"][:, 0, 4], r["final_state"][4])           # E constant
    for j in (1, 2, 3):
        rj = tab_oracle.integrate(tb, st, 0.01, 300 * j)
        assert np.array_equal(r["snapshots"][:, j, :], rj["final_state"].T)
    m = tab_oracle.integrate(tb, st, 0.01, 900, snapshot_every=100, snap_capacity=4, snap_mask=0x26)   # x1, x2, p1
    assert (m["snap_count"] == 10).all() and m["snapshots"].shape == (60, 4, 3)
    full = tab_oracle.integrate(tb, st, 0.01, 900, snapshot_every=100)
    assert np.array_equal(m["snapshots"], full["snapshots"][:, :4, [1, 2, 5]])
    # early termination: records stop with the particle
    out = st.copy()
    out[0] = 39.0
    out[3] = 2.0
    e = tab_oracle.integrate(tb, out, 0.05, 400, snapshot_every=5)
    assert (e["status"] == tab_oracle.ST_OUTSIDE).all()
    assert np.array_equal(e["snap_count"], 1 + e["steps_done"] // 5)
    for i in range(0, 60, 7):
        assert np.isnan(e["snapshots"][i, e["snap_count"][i]:]).all() and np.isfinite(e["snapshots"][i, : e["snap_count"][i]]).all()


def test_general_tabulated_trajectory_records(tab_oracle):
    """Records on the general path: the same S1-S3 semantics, pinned the same way (slot j == the shorter run, bitwise), and
    on an embedded eq.(8) table they are the five-field oracle's records (1e-12)."""
    a = 0.9
    tb5 = W.kerr_metric_table(1.0, a, 257, 65, 1.8, 40.0, 0.2, math.pi - 0.2)
    tb = W.general_table_from_diagonal(tb5)
    st = W.kerr_bound(40, a, W.SEED_BASE + 2)
    r = tab_oracle.integrate_general(tb, st, 0.01, 600, snapshot_every=200, snap_mask=0xFF)
    assert (r["snap_count"] == 4).all()
    assert np.array_equal(r["snapshots"][:, 0, [1, 2, 3, 5, 6, 7]], st.T)
    for j in (1, 3):
        rj = tab_oracle.integrate_general(tb, st, 0.01, 200 * j)
        assert np.array_equal(r["snapshots"][:, j, :], rj["final_state"].T)
    r5 = tab_oracle.integrate(tb5, st, 0.01, 600, snapshot_every=200)
    assert np.max(np.abs(r["snapshots"] - r5["snapshots"]) / np.maximum(np.abs(r5["snapshots"]), 1.0)) < 1e-12
    m = tab_oracle.integrate_general(tb, st, 0.01, 600, snapshot_every=100, snap_capacity=3, snap_mask=0x46)
    assert (m["snap_count"] == 7).all() and m["snapshots"].shape == (40, 3, 3)


# ---- reading T7: the adaptive RK5(4) stepper on the tabulated metric -----------------------------------------------------
def test_tabulated_adaptive_is_fifth_order_and_agrees_with_the_pinned_rk4_path(tab_oracle):
    """On the made-up metric with quadratic fields the interpolant is the metric itself (smooth), so with the controller
    off the propagated solution must converge with order 5 (Q -> 32; the pinned RK4 path gives 16); with the controller
    on it must land on the final time with the state the pinned fixed-step RK4 path reaches with a small step."""
    tb, _ = _quadratic_metric()
    rng = np.random.default_rng(9)
    n = 12
    st = np.stack([rng.uniform(1.6, 2.6, n), rng.uniform(1.2, 2.0, n), np.zeros(n), rng.uniform(-0.3, 0.3, n),
                   rng.uniform(-0.3, 0.3, n), rng.uniform(0.3, 1.0, n)])
    sols = []
    for k in (1, 2, 4):
        r = tab_oracle.integrate_adaptive(tb, st, 0.2 / k, np.inf, 1.0, 10**6, tau_end=2.0, long_double=True)
        assert (r["status"] == tab_oracle.ST_MAXSTEPS).all() and (r["steps_done"] == 10 * k).all() and (r["rejected"] == 0).all()
        sols.append(r["final_state"])
    Q = np.linalg.norm(sols[0] - sols[1], axis=0) / np.linalg.norm(sols[1] - sols[2], axis=0)
    assert Q.min() > 18.0 and abs(np.median(Q) - 32.0) < 6.0, Q
    ref = tab_oracle.integrate(tb, st, 0.0005, 4000, long_double=True)
    ad = tab_oracle.integrate_adaptive(tb, st, 0.1, 1e-11, 1e-11, 10**6, tau_end=2.0)
    assert np.max(np.abs(ad["final_state"] - ref["final_state"])) < 1e-9
    assert np.allclose(ad["final_state"][[4, 7]], ref["final_state"][[4, 7]], rtol=0, atol=1e-15)      # E, L constants


def test_tabulated_adaptive_kerr_converges_to_the_analytic_adaptive_oracle_and_stops_like_it(tab_oracle, oracle):
    a = 0.9
    st = W.kerr_bound(40, a, W.SEED_BASE + 2)
    ref = oracle.integrate_adaptive(oracle.KERR, 1.0, a, st, 0.05, 1e-10, 1e-10, 10**6, tau_end=30.0)
    errs = []
    for n1, n2 in ((513, 129), (1025, 257)):
        tb = W.kerr_metric_table(1.0, a, n1, n2, 1.8, 40.0, 0.2, math.pi - 0.2)
        r = tab_oracle.integrate_adaptive(tb, st, 0.05, 1e-10, 1e-10, 10**6, tau_end=30.0)
        assert (r["status"] == tab_oracle.ST_MAXSTEPS).all()
        errs.append(np.abs(r["final_state"][[1, 2, 5, 6]] - ref["final_state"][[1, 2, 5, 6]]).max())
    assert errs[1] < errs[0] / 3.0 and errs[1] < 2e-4, errs
    # stop rules: capture on a stage point, domain exit (T4), records stop with the particle, slot 0 = y0
    tb = W.kerr_metric_table(1.0, a, 257, 65, 1.8, 40.0, 0.2, math.pi - 0.2)
    out = st.copy()
    out[0] = 39.0
    out[3] = 2.0
    e = tab_oracle.integrate_adaptive(tb, out, 0.05, 1e-9, 1e-9, 10**5, snap_dtau=0.1, snap_capacity=50)
    assert (e["status"] == tab_oracle.ST_OUTSIDE).all() and (e["final_state"][1] <= 40.0).all()
    assert (e["snap_count"] >= 1).all() and np.array_equal(e["snapshots"][:, 0, [1, 2, 3, 5, 6, 7]], out.T)
    for i in range(0, 40, 7):
        cnt = e["snap_count"][i]
        assert np.isfinite(e["snapshots"][i, :cnt]).all() and np.isnan(e["snapshots"][i, cnt:]).all()
    inf = st.copy()
    inf[3] = -3.0                                   # thrown at the hole
    c = tab_oracle.integrate_adaptive(tb, inf, 0.05, 1e-9, 1e-9, 10**5, r_capture=2.5)
    assert (c["status"] == tab_oracle.ST_CAPTURED).all() and (c["final_state"][1] >= 2.5).all()
    # fixed-step mode: a record on a step boundary is that step's state
    f = tab_oracle.integrate_adaptive(tb, st, 0.25, np.inf, 1.0, 10**6, tau_end=3.0, snap_dtau=1.0, snap_capacity=5)
    assert (f["snap_count"] == 4).all()
    f2 = tab_oracle.integrate_adaptive(tb, st, 0.25, np.inf, 1.0, 10**6, tau_end=2.0)
    assert np.abs(f["snapshots"][:, 2, :] - f2["final_state"].T).max() < 1e-13


# ---- readings T6 + T7: the adaptive stepper on the GENERAL ten-field metric ----------------------------------------------
def test_general_adaptive_is_fifth_order_reduces_to_the_five_field_path_and_agrees_with_rk4(tab_oracle):
    """(i) On the made-up metric whose ten fields are all non-trivial quadratics (interpolant exact, smooth) the propagated
    solution converges with order 5 with the controller off (Q -> 32) and, with the controller on, lands on the state the
    PINNED fixed-step general RK4 path reaches with a small step.  (ii) On an embedded eq.(8) table the general adaptive
    oracle with the controller off agrees with the pinned five-field adaptive oracle to rounding, dense-output records
    included; with the controller on, at the tolerance's level."""
    tb, _ = _quadratic_general_metric()
    rng = np.random.default_rng(19)
    n = 12
    st = np.stack([rng.uniform(1.6, 2.6, n), rng.uniform(1.2, 2.0, n), np.zeros(n), rng.uniform(-0.3, 0.3, n),
                   rng.uniform(-0.3, 0.3, n), rng.uniform(0.3, 1.0, n)])
    sols = []
    for k in (1, 2, 4):
        r = tab_oracle.integrate_adaptive_general(tb, st, 0.2 / k, np.inf, 1.0, 10**6, tau_end=2.0, long_double=True)
        assert (r["status"] == tab_oracle.ST_MAXSTEPS).all() and (r["steps_done"] == 10 * k).all() and (r["rejected"] == 0).all()
        sols.append(r["final_state"])
    Q = np.linalg.norm(sols[0] - sols[1], axis=0) / np.linalg.norm(sols[1] - sols[2], axis=0)
    assert Q.min() > 18.0 and abs(np.median(Q) - 32.0) < 6.0, Q
    ref = tab_oracle.integrate_general(tb, st, 0.0005, 4000, long_double=True)
    ad = tab_oracle.integrate_adaptive_general(tb, st, 0.1, 1e-11, 1e-11, 10**6, tau_end=2.0)
    assert np.max(np.abs(ad["final_state"] - ref["final_state"])) < 1e-9
    assert np.allclose(ad["final_state"][[4, 7]], ref["final_state"][[4, 7]], rtol=0, atol=1e-15)      # E, L constants
    # (ii)
    a = 0.9
    tb5 = W.kerr_metric_table(1.0, a, 257, 65, 1.8, 40.0, 0.2, math.pi - 0.2)
    tb10 = W.general_table_from_diagonal(tb5)
    sk = W.kerr_bound(40, a, W.SEED_BASE + 2)
    kw = dict(tau_end=30.0, snap_dtau=2.5, snap_capacity=13)
    r5 = tab_oracle.integrate_adaptive(tb5, sk, 0.05, np.inf, 1.0, 10**6, **kw)          # controller off: same step sequence
    r10 = tab_oracle.integrate_adaptive_general(tb10, sk, 0.05, np.inf, 1.0, 10**6, **kw)
    assert np.array_equal(r5["status"], r10["status"]) and np.array_equal(r5["steps_done"], r10["steps_done"])
    assert (r5["steps_done"] == 600).all() and np.array_equal(r5["snap_count"], r10["snap_count"]) and (r5["snap_count"] == 13).all()
    assert np.max(np.abs(r5["final_state"] - r10["final_state"]) / np.maximum(np.abs(r5["final_state"]), 1.0)) < 1e-11
    assert np.max(np.abs(r5["snapshots"] - r10["snapshots"]) / np.maximum(np.abs(r5["snapshots"]), 1.0)) < 1e-11
    # controller on: on a C^1 interpolant the accept / reject decisions are sensitive to rounding, the step
    # sequences differ; what the tolerance determines -- the state at tau_end -- agrees at the tolerance's level
    a5 = tab_oracle.integrate_adaptive(tb5, sk, 0.05, 1e-9, 1e-9, 10**6, tau_end=30.0)
    a10 = tab_oracle.integrate_adaptive_general(tb10, sk, 0.05, 1e-9, 1e-9, 10**6, tau_end=30.0)
    assert np.array_equal(a5["status"], a10["status"])
    assert np.max(np.abs(a5["final_state"] - a10["final_state"]) / np.maximum(np.abs(a5["final_state"]), 1.0)) < 2e-5      # measured 2.3e-6


def test_general_adaptive_kerr_schild_matches_the_analytic_boyer_lindquist_oracle_and_follows_a_plunge(tab_oracle, oracle):
    """Kerr a = 0.9 in ingoing Kerr-Schild coordinates on a ten-field table, adaptive: (r, theta, p_theta) of bound orbits
    at tau = 30 converge to the ANALYTIC adaptive Boyer-Lindquist oracle with the grid; a particle thrown at the hole is
    followed THROUGH the horizon (capture radius inside r_+) with finite state; domain exit and capture semantics (T4, T7)."""
    a, M = 0.9, 1.0
    st, consts = W.kerr_bound(40, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_kerr_schild(st, consts[0], M, a)
    ref = oracle.integrate_adaptive(oracle.KERR, M, a, st, 0.05, 1e-10, 1e-10, 10**6, tau_end=30.0)
    errs = []
    for n1, n2 in ((513, 129), (1025, 257)):
        tb = W.kerr_schild_metric_table(M, a, n1, n2, 1.2, 40.0, 0.15, math.pi - 0.15)
        r = tab_oracle.integrate_adaptive_general(tb, ks, 0.05, 1e-10, 1e-10, 10**6, tau_end=30.0)
        assert (r["status"] == tab_oracle.ST_MAXSTEPS).all()
        errs.append(np.abs(r["final_state"][[1, 2, 6]] - ref["final_state"][[1, 2, 6]]).max())
        assert np.max(np.abs(r["final_state"][4] - consts[0])) < 1e-4          # E of the interpolated metric's mass shell
    assert errs[1] < errs[0] / 3.0 and errs[1] < 2e-4, errs
    rp = M + math.sqrt(M * M - a * a)
    tb = W.kerr_schild_metric_table(M, a, 513, 129, 1.1, 40.0, 0.15, math.pi - 0.15)
    fall = np.zeros((6, 8))
    fall[0] = np.linspace(5.0, 8.0, 8)
    fall[1] = np.linspace(0.8, 2.2, 8)
    fall[3] = -0.2
    fall[5] = np.linspace(-1.0, 1.0, 8)
    c = tab_oracle.integrate_adaptive_general(tb, fall, 0.05, 1e-9, 1e-9, 10**5, r_capture=1.25, snap_dtau=1.0, snap_capacity=200)
    assert (c["status"] == tab_oracle.ST_CAPTURED).all() and (c["final_state"][1] >= 1.25).all() and (c["final_state"][1] < rp).all()
    assert np.isfinite(c["final_state"]).all() and (c["health"] < 1e-4).all()
    for i in range(8):
        cnt = c["snap_count"][i]
        assert cnt >= 2 and np.isfinite(c["snapshots"][i, :cnt]).all() and np.isnan(c["snapshots"][i, cnt:]).all()
    out = ks.copy()
    out[0] = 39.0
    out[3] = 2.0
    e = tab_oracle.integrate_adaptive_general(tb, out, 0.05, 1e-9, 1e-9, 10**5)
    assert (e["status"] == tab_oracle.ST_OUTSIDE).all() and (e["final_state"][1] <= 40.0).all()
