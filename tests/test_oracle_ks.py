"""Pins of the Cartesian Kerr-Schild oracle (oracle/geo_ks_oracle.cpp; SURVEY 8(f).3 second clause, DESIGN.md readings
K1-K5) to what the paper and the mathematics fix -- not to itself.  CPU only (``-m "not gpu"``).

* the metric: g = eta + f l l pulled back through the coordinate map equals the paper's metric (6),
  entry by entry -- fixes f, l_mu, r(x, y, z) and the sign of a;
* the right-hand side: 40-digit differentiation of H = 1/2 g^{mu nu} p_mu p_nu (eqs.(3),(4) PAPER.md:60-65) with g^{mu nu}
  from the numerically inverted 4 x 4 matrix -- no derivative formula shared with the oracle; points next to the polar
  axis and inside the horizon included;
* the 3+1 split (line element (1) PAPER.md:47) and the mass shell (5) by numerical inversion of gamma_ij;
* dynamics: orbits of the PINNED Boyer-Lindquist oracle transformed into this chart agree at common tau in the
  quantities the charts share (r, cos theta, E, L_z, Carter's Q) and converge at fourth order;
* M = 0: exact straight lines; a tilted Schwarzschild circle keeps r and crosses z = 0 at that r (reading K3);
* where the Boyer-Lindquist chart cannot go -- through the polar axis and through the horizon -- L_z, Q and 2H stay
  constant to O(h^4);
* stop rules and records: the readings' semantics on hand-made cases, slot j == final state of the shorter run (bitwise).
"""
import math
import os
import sys

import mpmath as mp
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "oracle"))

import geo_ks_oracle as KS  # noqa: E402
import geo_oracle as BL  # noqa: E402
from paper_1803_08320_b200 import workloads as W  # noqa: E402

NCPU = min(os.cpu_count() or 1, 16)


# ---------------------------------------------------------------------------
# definitions typed from the literature (Kerr 1963; Kerr & Schild 1965), in mpmath / numpy
# ---------------------------------------------------------------------------
def _ks_g_mp(M, a, x, y, z):
    w = x * x + y * y + z * z - a * a
    r = mp.sqrt((w + mp.sqrt(w * w + 4 * a * a * z * z)) / 2)
    f = 2 * M * r ** 3 / (r ** 4 + a * a * z * z)
    l = mp.matrix([1, (r * x + a * y) / (r * r + a * a), (r * y - a * x) / (r * r + a * a), z / r])
    g = mp.diag([-1, 1, 1, 1]) + f * (l * l.T)
    return g


def _H_mp(M, a, x, y, z, pt_std, px, py, pz):
    ginv = mp.inverse(_ks_g_mp(M, a, x, y, z))
    p = mp.matrix([pt_std, px, py, pz])
    return (p.T * ginv * p)[0] / 2


def _rhs_by_differentiation(M, a, y8):
    mp.mp.dps = 40
    t, x, y, z, E, px, py, pz = [mp.mpf(float(v)) for v in y8]
    M, a = mp.mpf(M), mp.mpf(a)
    H = lambda X, Y, Z, PT, PX, PY, PZ: _H_mp(M, a, X, Y, Z, PT, PX, PY, PZ)   # noqa: E731
    at = (x, y, z, -E, px, py, pz)
    d = lambda k: mp.diff(H, at, tuple(1 if j == k else 0 for j in range(7)))   # noqa: E731
    # xdot^mu = dH/dp_mu, pdot_i = -dH/dx^i  (eq.(3))
    return [float(v) for v in (d(3), d(4), d(5), d(6), -d(0), -d(1), -d(2))]


def _metric6_np(M, a, r, th):
    """Metric (6) PAPER.md:73-84, order (t, r, theta, phi)."""
    s, c = math.sin(th), math.cos(th)
    rho2 = r * r + a * a * c * c
    Delta = r * r - 2 * M * r + a * a
    Sigma = (r * r + a * a) ** 2 - a * a * Delta * s * s
    g = np.zeros((4, 4))
    g[0, 0] = -(Delta - a * a * s * s) / rho2
    g[0, 3] = g[3, 0] = -2 * a * M * r * s * s / rho2
    g[1, 1] = rho2 / Delta
    g[2, 2] = rho2
    g[3, 3] = Sigma * s * s / rho2
    return g


def _map_bl_to_ks(a, r, th, ph):
    s, c = math.sin(th), math.cos(th)
    return ((r * math.cos(ph) - a * math.sin(ph)) * s, (r * math.sin(ph) + a * math.cos(ph)) * s, r * c)


# ---------------------------------------------------------------------------
# the metric
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("a", [0.0, 0.5, -0.7, 0.998])
def test_metric_is_paper_metric6_pulled_back(a):
    """J^T (eta + f l l) J = metric (6), J = d(t~, x, y, z)/d(t, r, theta, phi) with dt~ = dt + 2Mr/Delta dr,
    dphi~ = dphi + a/Delta dr, x + iy = (r + ia) sin(theta) e^{i phi~}, z = r cos(theta)."""
    M = 1.0
    rng = np.random.default_rng(5)
    for _ in range(40):
        r = rng.uniform(2.1, 30.0)
        th = rng.uniform(0.05, math.pi - 0.05)
        ph = rng.uniform(-3.0, 3.0)
        s, c = math.sin(th), math.cos(th)
        sp, cp = math.sin(ph), math.cos(ph)
        Delta = r * r - 2 * M * r + a * a
        x, y, z = _map_bl_to_ks(a, r, th, ph)
        f, lx, ly, lz = KS.metric(M, a, x, y, z)
        l = np.array([1.0, lx, ly, lz])
        g_ks = np.diag([-1.0, 1.0, 1.0, 1.0]) + f * np.outer(l, l)
        dx_dr, dx_dth, dx_dph = cp * s, (r * cp - a * sp) * c, -y
        dy_dr, dy_dth, dy_dph = sp * s, (r * sp + a * cp) * c, x
        J = np.zeros((4, 4))          # J[mu][b]: new coordinate mu, BL coordinate b
        J[0, 0] = 1.0
        J[0, 1] = 2 * M * r / Delta
        J[1, 1] = dx_dr + dx_dph * a / Delta
        J[1, 2] = dx_dth
        J[1, 3] = dx_dph
        J[2, 1] = dy_dr + dy_dph * a / Delta
        J[2, 2] = dy_dth
        J[2, 3] = dy_dph
        J[3, 1] = c
        J[3, 2] = -r * s
        g_bl = J.T @ g_ks @ J
        ref = _metric6_np(M, a, r, th)
        scale = np.sqrt(np.abs(np.outer(np.diag(ref), np.diag(ref))))
        assert np.max(np.abs(g_bl - ref) / scale) < 5e-12, (a, r, th, np.max(np.abs(g_bl - ref) / scale))
        assert abs(KS.radius(M, a, x, y, z) - r) < 1e-12 * r


def test_radius_is_the_spheroid_root_and_regular_on_the_axis():
    M, a = 1.0, 0.9
    for (x, y, z) in [(0.0, 0.0, 3.0), (0.0, 0.0, -0.4), (1e-200, 0.0, 2.0), (3.0, 4.0, 0.0), (0.3, -0.2, 1e-9)]:
        r = KS.radius(M, a, x, y, z)
        assert r >= 0
        if r > 0:
            assert abs((x * x + y * y) / (r * r + a * a) + z * z / (r * r) - 1.0) < 1e-12
    assert KS.radius(M, a, 0.0, 0.0, 3.0) == pytest.approx(3.0, rel=1e-15)          # on the axis r = |z|
    assert KS.radius(M, a, 3.0, 4.0, 0.0) == pytest.approx(math.sqrt(25.0 - 0.81), rel=1e-15)   # equator: r^2 = R^2 - a^2


# ---------------------------------------------------------------------------
# the right-hand side
# ---------------------------------------------------------------------------
def _random_states(seed, n, a):
    rng = np.random.default_rng(seed)
    out = []
    for k in range(n):
        if k % 4 == 0:      # next to the polar axis
            x, y, z = rng.uniform(-1e-3, 1e-3), rng.uniform(-1e-3, 1e-3), rng.uniform(1.5, 8.0) * rng.choice([-1, 1])
        elif k % 4 == 1:    # inside the horizon, away from the ring
            x, y, z = rng.uniform(-0.6, 0.6), rng.uniform(-0.6, 0.6), rng.uniform(0.5, 0.9) * rng.choice([-1, 1])
        else:
            x, y, z = rng.uniform(-12, 12), rng.uniform(-12, 12), rng.uniform(-12, 12)
        p = rng.uniform(-1.5, 1.5, 3)
        E = rng.uniform(0.5, 1.5)
        out.append([rng.uniform(0, 5), x, y, z, E, p[0], p[1], p[2]])
    return out


@pytest.mark.parametrize("a", [0.0, 0.6, -0.9, 0.998])
def test_rhs_matches_high_precision_differentiation_of_H(a):
    """Hamilton's equations (3),(4) PAPER.md:60-65: every component of the oracle's RHS against mp.diff of
    H = 1/2 p g^{-1} p with g^{-1} from mp.inverse of eta + f l l."""
    M = 1.0
    worst = 0.0
    for y8 in _random_states(11 + int(abs(a) * 100), 16, a):
        ref = np.array(_rhs_by_differentiation(M, a, y8))
        got = KS.rhs(M, a, y8)
        got_ld = KS.rhs(M, a, y8, long_double=True)
        scale = np.maximum(np.abs(ref), 1e-3 * np.max(np.abs(ref)))
        worst = max(worst, float(np.max(np.abs(got - ref) / scale)))
        assert np.max(np.abs(got - ref) / scale) < 2e-10, (y8, got, ref)      # cancellation next to the axis costs digits
        assert np.max(np.abs(got_ld - ref) / scale) < 2e-13, (y8, got_ld, ref)
    assert worst > 0.0


def test_hamiltonian_matches_inverted_matrix():
    M, a = 1.0, 0.8
    mp.mp.dps = 40
    for y8 in _random_states(3, 12, a):
        ref = float(_H_mp(mp.mpf(M), mp.mpf(a), *[mp.mpf(float(v)) for v in (y8[1], y8[2], y8[3], -y8[4], y8[5], y8[6], y8[7])]))
        assert KS.hamiltonian(M, a, y8) == pytest.approx(ref, rel=1e-11, abs=1e-12)


def test_3p1_split_and_mass_shell():
    """Line element (1) PAPER.md:47 read off g = eta + f l l: gamma_ij = g_ij, beta_i = g_ti, alpha^2 = beta_i beta^i - g_tt,
    with gamma^{ij} by numpy inversion; the oracle's E solves 2H = -kappa (eq.(5)) as the future-directed root
    E = alpha sqrt(kappa + gamma^{ij} p_i p_j) - beta^k p_k."""
    M, a = 1.0, 0.9
    for y8 in _random_states(21, 24, a):
        x, y, z = y8[1:4]
        p = np.array(y8[5:8])
        f, lx, ly, lz = KS.metric(M, a, x, y, z)
        l = np.array([lx, ly, lz])
        gam = np.eye(3) + f * np.outer(l, l)
        beta_lo = f * l
        gam_inv = np.linalg.inv(gam)
        beta_up = gam_inv @ beta_lo
        alpha2 = beta_lo @ beta_up - (-1.0 + f)
        assert alpha2 == pytest.approx(1.0 / (1.0 + f), rel=1e-12)
        for kappa in (0.0, 1.0):
            E_ref = math.sqrt(alpha2 * (kappa + p @ gam_inv @ p)) - beta_up @ p
            E = KS.energy(M, a, x, y, z, p[0], p[1], p[2], kappa)
            assert E == pytest.approx(E_ref, rel=1e-12, abs=1e-13)
            yE = list(y8)
            yE[4] = E
            assert 2.0 * KS.hamiltonian(M, a, yE) + kappa == pytest.approx(0.0, abs=1e-11 * max(1.0, E * E))


def test_energy_is_the_boyer_lindquist_energy_of_the_same_covector():
    """p_t is the same number in both charts (dt~ = dt + ... dr): the mass-shell E of transformed data equals the pinned
    Boyer-Lindquist oracle's E."""
    M, a = 1.0, 0.9
    st, consts = W.kerr_bound(64, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, consts[0], M, a)
    for i in range(64):
        E_bl = BL.energy(M, a, st[0, i], st[1, i], st[3, i], st[4, i], st[5, i], 1.0)
        E_ks = KS.energy(M, a, *ks[:, i], 1.0)
        assert E_ks == pytest.approx(E_bl, rel=2e-13)
        assert ks[0, i] * ks[4, i] - ks[1, i] * ks[3, i] == pytest.approx(st[5, i], rel=1e-12, abs=1e-12)   # L_z = x p_y - y p_x


# ---------------------------------------------------------------------------
# dynamics against the pinned Boyer-Lindquist oracle
# ---------------------------------------------------------------------------
def _shared(fin_ks, a, kappa):
    """(r, cos theta, E, L_z, Q) from a Cartesian Kerr-Schild record [8][n]; Q = p_theta^2 + cos^2 (a^2 (kappa - E^2) + L_z^2/sin^2),
    p_theta = sum_i dx^i/dtheta p_i = cot(theta) (x p_x + y p_y) - r sin(theta) p_z."""
    t, x, y, z, E, px, py, pz = fin_ks
    r = W.kerr_schild_radius(np.stack([x, y, z]), a)
    c = z / r
    s = np.sqrt(1.0 - c * c)
    Lz = x * py - y * px
    pth = c / s * (x * px + y * py) - r * s * pz
    Q = pth ** 2 + c * c * (a * a * (kappa - E * E) + Lz * Lz / (s * s))
    return r, c, E, Lz, Q


def test_bound_orbits_match_the_boyer_lindquist_oracle_and_converge():
    """Kerr a = 0.9 bound orbits (the config-2 distribution): r, cos(theta) at tau = 40 against the pinned Boyer-Lindquist
    oracle on the same geodesics; the difference is the two RK4 truncation errors and falls ~16x per halving of h."""
    M, a = 1.0, 0.9
    st, consts = W.kerr_bound(96, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, consts[0], M, a)
    errs = []
    for h, n in [(0.04, 1000), (0.02, 2000), (0.01, 4000)]:
        ob = BL.integrate(BL.KERR, M, a, st, h, n, nthreads=NCPU)
        ok = KS.integrate(M, a, ks, h, n, nthreads=NCPU)
        r, c, E, Lz, Q = _shared(ok["final_state"], a, 1.0)
        e_r = np.max(np.abs(r - ob["final_state"][1]) / ob["final_state"][1])
        e_c = np.max(np.abs(c - np.cos(ob["final_state"][2])))
        errs.append(max(e_r, e_c))
        assert np.all(ok["status"] == KS.ST_MAXSTEPS) and np.all(ok["steps_done"] == n)
        assert np.max(np.abs(E - consts[0])) < 1e-13 and np.max(np.abs(Lz - consts[1])) < 1e-6
    assert errs[2] < 2e-9, errs
    assert errs[0] / errs[1] > 8 and errs[1] / errs[2] > 8, errs          # fourth order (16x) with margin


def test_constants_of_motion_converge_at_fourth_order():
    """L_z (NOT a momentum of this chart), Carter's Q and 2H drift as O(h^4): ratio ~16 per halving (long double, so the
    drift is truncation, not rounding)."""
    M, a = 1.0, 0.9
    st, consts = W.kerr_bound(48, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, consts[0], M, a)
    drift = []
    for h, n in [(0.2, 500), (0.1, 1000), (0.05, 2000)]:
        o = KS.integrate(M, a, ks, h, n, long_double=True, nthreads=NCPU)
        r, c, E, Lz, Q = _shared(o["final_state"], a, 1.0)
        drift.append([np.max(np.abs(Lz - consts[1])), np.max(np.abs(Q - consts[2]) / (1 + consts[2])), np.max(o["health"])])
    drift = np.array(drift)
    assert np.all(drift[2] < 1e-7), drift
    assert np.all(drift[0] / drift[1] > 8) and np.all(drift[1] / drift[2] > 8), drift


def test_flat_space_straight_lines():
    """M = 0 (f = 0; the spheroidal r still carries a): x(tau) = x0 + p tau exactly, t~ = E tau, E = sqrt(kappa + p^2)."""
    rng = np.random.default_rng(7)
    n = 32
    st = np.vstack([rng.uniform(-5, 5, (3, n)), rng.uniform(-1, 1, (3, n))])
    for kind, kappa in ((KS.TIMELIKE, 1.0), (KS.NULL, 0.0)):
        o = KS.integrate(0.0, 0.7, st, 0.125, 800, kind=kind)
        tau = 100.0
        fin = o["final_state"]
        assert np.max(np.abs(fin[1:4] - (st[0:3] + tau * st[3:6]))) < 1e-12
        assert np.max(np.abs(fin[5:8] - st[3:6])) == 0.0
        E = np.sqrt(kappa + (st[3:6] ** 2).sum(0))
        assert np.max(np.abs(fin[4] - E)) < 1e-15 and np.max(np.abs(fin[0] - E * tau)) < 1e-11


def test_tilted_schwarzschild_circle_and_equatorial_event():
    """a = 0: a circular orbit of radius R in a plane tilted by 40 degrees (closed form: L^2 = M R^2/(R - 3M), eq.(34)
    family; E^2 = (R - 2M)^2 / (R (R - 3M))): r(x, y, z) stays R, E matches, and the first crossing of z = 0 is reported at
    r = R (reading K3: linear in z between the bracketing states; both have r = R)."""
    M, R, inc = 1.0, 8.0, math.radians(40.0)
    L = math.sqrt(M * R * R / (R - 3 * M))
    E = (R - 2 * M) / math.sqrt(R * (R - 3 * M))
    # isotropic-free construction: at a = 0 the spatial covector of a circular orbit is tangential with |p| = L / R
    # (p_r~ = 2 M E/(R - 2M) from the ingoing time: p_r~ = p_r + 2 M r E / Delta with p_r = 0)
    e_r = np.array([math.cos(0.3), math.sin(0.3) * math.cos(inc), math.sin(0.3) * math.sin(inc)])
    e_t = np.array([-math.sin(0.3), math.cos(0.3) * math.cos(inc), math.cos(0.3) * math.sin(inc)])
    pos = R * e_r
    p = (L / R) * e_t + (2 * M * E / (R - 2 * M)) * e_r
    st = np.concatenate([pos, p])[:, None]
    T = 2 * math.pi * math.sqrt(R ** 3 / M) * math.sqrt(1 - 3 * M / R)       # proper-time period
    h = 0.01
    n = int(0.75 * T / h)
    o = KS.integrate(M, 0.0, st, h, n, snapshot_every=50)
    assert o["final_state"][4, 0] == pytest.approx(E, rel=1e-13)
    snaps = o["snapshots"][0, :o["snap_count"][0]]
    rr = np.sqrt((snaps[:, 1:4] ** 2).sum(1))
    assert np.max(np.abs(rr - R)) < 1e-9
    assert o["eq_cross_r"][0] == pytest.approx(R, rel=1e-9)
    # orbital phase after tau: angle from the start direction = sqrt(M/R^3)/sqrt(1 - 3M/R) tau
    ang = math.atan2(snaps[-1, 1:4] @ e_t, snaps[-1, 1:4] @ e_r) % (2 * math.pi)
    tau = h * 50 * (len(snaps) - 1)
    assert ang == pytest.approx((2 * math.pi * tau / T) % (2 * math.pi), abs=2e-9)


def _axis_and_plunge_states(a):
    """(i) timelike particles aimed THROUGH the polar axis (x = y = 0 is hit, or missed by <= 1e-6, at mid-flight) -- a
    place where the Boyer-Lindquist chart of eq.(6) is singular; (ii) particles dropped into the hole."""
    n = 12
    st = np.zeros((6, n))
    for k in range(6):
        off = 0.0 if k < 3 else 1e-6 * k
        st[:, k] = [-6.0, off, 7.0 + 0.5 * k, 1.2, 0.0, 0.05 * k]         # moving in +x towards the axis above the hole (unbound)
    for k in range(6, n):
        j = k - 6
        st[:, k] = [7.0 + 0.3 * j, 1.0, 0.5 * (j - 2), -0.4, 0.03 * j, 0.0]      # infall with some L_z
    return st


@pytest.mark.parametrize("a", [0.9, 0.998])
def test_polar_axis_and_horizon_are_regular(a):
    M = 1.0
    st = _axis_and_plunge_states(a)
    rp = M + math.sqrt(M * M - a * a)
    E0 = np.array([KS.energy(M, a, *st[:, i], 1.0) for i in range(st.shape[1])])
    Lz0 = st[0] * st[4] - st[1] * st[3]
    o = KS.integrate(M, a, st, 0.01, 6000, r_capture=0.9 * rp, r_escape=200.0, snapshot_every=100, nthreads=NCPU)
    assert np.all(o["status"][:6] == KS.ST_MAXSTEPS)            # the axis crossers fly by
    assert np.all(o["status"][6:] == KS.ST_CAPTURED)            # the others end INSIDE the horizon
    fin = o["final_state"]
    r_fin = W.kerr_schild_radius(fin[1:4], a)
    assert np.all(r_fin[6:] < rp) and np.all(np.isfinite(fin))
    assert np.max(o["health"][:6]) < 1e-10 and np.max(o["health"][6:]) < 1e-5      # O(h^4), largest for the grazing infall
    assert np.max(np.abs(fin[4] - E0)) == 0.0
    dLz = np.abs(fin[1] * fin[6] - fin[2] * fin[5] - Lz0)
    assert np.max(dLz[:6]) < 1e-10 and np.max(dLz[6:]) < 1e-5
    # the axis crossers really pass through the axis: L_z = 0 (or ~1e-6), and the distance from the axis falls below one
    # step length (records of every step of the first 1500)
    dense = KS.integrate(M, a, st[:, :6], 0.01, 1500, snapshot_every=1, snap_mask=0x0E)
    rho = np.sqrt(dense["snapshots"][:, :, 0] ** 2 + dense["snapshots"][:, :, 1] ** 2)
    assert np.all(rho.min(axis=1) < 0.012), rho.min(axis=1)
    assert np.all(dense["snapshots"][:, 0, 0] < 0) and np.all(dense["snapshots"][:, -1, 0] > 0)
    # Carter's constant before / after the axis passage (evaluated off the axis)
    y0 = np.vstack([np.zeros(6), st[0:3, :6], E0[:6], st[3:6, :6]])
    Q0 = _shared(y0, a, 1.0)[4]
    Q1 = _shared(fin[:, :6], a, 1.0)[4]
    assert np.max(np.abs(Q1 - Q0) / (1 + np.abs(Q0))) < 1e-9


# ---------------------------------------------------------------------------
# stop rules and records
# ---------------------------------------------------------------------------
def test_stop_rules_and_records():
    M, a = 1.0, 0.9
    st = _axis_and_plunge_states(a)[:, 6:]
    n = st.shape[1]
    full = KS.integrate(M, a, st, 0.02, 3000, r_capture=1.6, r_escape=50.0, snapshot_every=25, snap_mask=0x6F)
    r_fin = W.kerr_schild_radius(full["final_state"][1:4], a)
    assert np.all(full["status"] == KS.ST_CAPTURED)
    assert np.all(r_fin >= 1.6)                                   # B2: the capturing step is not taken
    # one more step from the final state leaves the domain at one of its evaluation points
    nxt = KS.integrate(M, a, np.vstack([full["final_state"][1:4], full["final_state"][5:8]]), 0.02, 1, r_capture=-np.inf)
    assert np.all(W.kerr_schild_radius(nxt["final_state"][1:4], a) < 1.6 + 0.02)
    assert np.all(full["snap_count"] == 1 + full["steps_done"] // 25)                       # S1
    # slot j == final state of the run that stops after 25 j steps (bitwise), masked components (t,x,y,z,px,py)
    for j in (1, 3):
        short = KS.integrate(M, a, st, 0.02, 25 * j, r_capture=1.6, r_escape=50.0)
        ok = full["steps_done"] >= 25 * j
        assert ok.any()
        comp = short["final_state"][[0, 1, 2, 3, 5, 6]][:, ok].T
        assert np.array_equal(full["snapshots"][ok, j, :], comp)
    # B1: a start inside the capture radius / beyond the escape radius ends at once with 0 steps; S3: capacity
    st2 = st.copy()
    st2[0:3, 0] = [0.5, 0.2, 0.3]
    st2[0:3, 1] = [80.0, 0.0, 1.0]
    o = KS.integrate(M, a, st2, 0.02, 100, r_capture=1.6, r_escape=50.0, snapshot_every=10, snap_capacity=3)
    assert o["status"][0] == KS.ST_CAPTURED and o["steps_done"][0] == 0 and o["snap_count"][0] == 0
    assert o["status"][1] == KS.ST_ESCAPED and o["steps_done"][1] == 0 and o["snap_count"][1] == 1
    assert np.all(o["snap_count"][2:] == 1 + o["steps_done"][2:] // 10) and o["snapshots"].shape[1] == 3
    # the ring singularity with the capture test disabled: non-finite, never a hang (B6 / NaN r counts as captured)
    ring = np.array([[a + 1e-3], [0.0], [1e-4], [-0.5], [0.0], [-0.05]])
    o = KS.integrate(M, a, ring, 0.05, 2000, r_capture=-np.inf)
    assert o["status"][0] in (KS.ST_NUMERIC, KS.ST_CAPTURED, KS.ST_MAXSTEPS)
    # plain update flag differs from Kahan only by rounding
    p = KS.integrate(M, a, st, 0.02, 500, flags=KS.FLAG_PLAIN_UPDATE)
    k = KS.integrate(M, a, st, 0.02, 500)
    d = np.max(np.abs(p["final_state"] - k["final_state"]))
    assert 0 < d < 1e-8


# ---------------------------------------------------------------------------
# reading K6: the adaptive RK5(4) stepper in this chart
# ---------------------------------------------------------------------------
def test_adaptive_is_fifth_order_and_lands_on_the_pinned_fixed_step_solution():
    """Controller off (rtol = inf): the propagated solution converges with order 5 (Q ~ 32-50 on these orbits at h = 1, 1/2, 1/4; the pinned RK4 path gives 16).
    Controller on: it lands on tau_end with the state the PINNED fixed-step path of this file reaches with a small step;
    E is untouched, L_z (not a momentum of the chart) is conserved to the tolerance."""
    M, a = 1.0, 0.9
    st, consts = W.kerr_bound(24, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, consts[0], M, a)
    sols = []
    for k in (1, 2, 4):
        r = KS.integrate_adaptive(M, a, ks, 1.0 / k, np.inf, 1.0, 10**6, tau_end=40.0, long_double=True)
        assert (r["status"] == KS.ST_MAXSTEPS).all() and (r["steps_done"] == 40 * k).all() and (r["rejected"] == 0).all()
        sols.append(r["final_state"])
    d12 = np.linalg.norm(sols[1] - sols[2], axis=0)
    big = d12 > 1e-12                      # above the rounding of the double-precision output
    Q = np.linalg.norm(sols[0] - sols[1], axis=0)[big] / d12[big]
    # the ratio scatters per orbit (the leading error term changes sign along an orbit); a fourth-order pair would give 16
    assert big.sum() >= 10 and Q.min() > 17.0 and 28.0 < np.median(Q) < 64.0, Q
    ref = KS.integrate(M, a, ks, 0.0025, 4000, long_double=True, nthreads=NCPU)
    ad = KS.integrate_adaptive(M, a, ks, 0.1, 1e-12, 1e-12, 10**6, tau_end=10.0, nthreads=NCPU)
    assert (ad["status"] == KS.ST_MAXSTEPS).all() and (ad["rejected"] >= 0).all()
    assert np.max(np.abs(ad["final_state"] - ref["final_state"]) / np.maximum(np.abs(ref["final_state"]), 1.0)) < 1e-9
    assert np.max(np.abs(ad["final_state"][4] - ref["final_state"][4])) < 4e-16            # E: constant (ref ran in long double)
    f = ad["final_state"]
    assert np.max(np.abs(f[1] * f[6] - f[2] * f[5] - consts[1])) < 1e-9


def test_adaptive_matches_the_boyer_lindquist_adaptive_oracle_and_dense_records():
    """Bound orbits to tau = 40 at a tight tolerance: r, cos(theta) equal those of the pinned Boyer-Lindquist adaptive oracle
    (another chart, another right-hand side) to the tolerance.  Dense output (A3): records at tau_j = 2.5 j equal the
    fixed-step path's states at the same tau to the continuous extension's accuracy; record 0 = y0; in fixed-step mode a
    record on a step boundary is that step's state."""
    M, a = 1.0, 0.9
    st, consts = W.kerr_bound(40, a, W.SEED_BASE + 2, return_constants=True)
    ks = W.to_cartesian_kerr_schild(st, consts[0], M, a)
    bl = BL.integrate_adaptive(BL.KERR, M, a, st, 0.05, 1e-12, 1e-12, 10**6, tau_end=40.0, nthreads=NCPU)
    ad = KS.integrate_adaptive(M, a, ks, 0.05, 1e-12, 1e-12, 10**6, tau_end=40.0, snap_dtau=2.5, snap_capacity=17, nthreads=NCPU)
    r, c, E, Lz, Q = _shared(ad["final_state"], a, 1.0)
    assert np.max(np.abs(r - bl["final_state"][1]) / bl["final_state"][1]) < 2e-9
    assert np.max(np.abs(c - np.cos(bl["final_state"][2]))) < 2e-9
    assert (ad["snap_count"] == 17).all()
    assert np.array_equal(ad["snapshots"][:, 0, [1, 2, 3, 5, 6, 7]], ks.T) and np.all(ad["snapshots"][:, 0, 0] == 0.0)
    fx = KS.integrate(M, a, ks, 0.0025, 16000, snapshot_every=1000, long_double=True, nthreads=NCPU)
    e = np.abs(ad["snapshots"] - fx["snapshots"]) / np.maximum(np.abs(fx["snapshots"]), 1.0)
    assert e.max() < 1e-8, e.max()
    f = KS.integrate_adaptive(M, a, ks, 0.25, np.inf, 1.0, 10**6, tau_end=3.0, snap_dtau=1.0, snap_capacity=5)
    f2 = KS.integrate_adaptive(M, a, ks, 0.25, np.inf, 1.0, 10**6, tau_end=2.0)
    assert (f["snap_count"] == 4).all() and np.abs(f["snapshots"][:, 2, :] - f2["final_state"].T).max() < 1e-13


def test_adaptive_camera_rays_get_every_class_right_where_both_fixed_step_charts_fail():
    """configs[2] rays (a = 0.998, i = 60 deg) with step control, rtol = atol = 1e-9: the termination class equals the
    closed-form capture criterion on EVERY ray of (i) the 10 polar-axis columns (64 rows), where the fixed-step
    Boyer-Lindquist path fails (reading B7), and (ii) the pixels at the prograde edge of the shadow where the fixed-step path
    of this chart fails, and (iii) a strided sub-image; |2H| of the escaped rays stays at the tolerance's level
    (readings K6a, K6b are what makes this work: step cap r/4, capture test on end points only)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from test_gpu_fullsize import _escapes_analytic
    M, a, N = 1.0, 0.998, 1024
    rp = W.horizon_radius(M, a)
    full, consts = W.camera_rays(N, a, 60.0, return_constants=True)
    img = np.arange(N * N).reshape(N, N)
    sel = np.concatenate([img[8::16, N // 2 - 5:N // 2 + 5].ravel(), img[440:600:2, 386:392].ravel(), img[32::64, 32::64].ravel()])
    st = np.ascontiguousarray(full[:, sel])
    ks = W.to_cartesian_kerr_schild(st, np.ones(len(sel)), M, a)
    o = KS.integrate_adaptive(M, a, ks, 0.02, 1e-9, 1e-9, 200000, r_capture=rp + 0.01, r_escape=1100.0, kind=KS.NULL, nthreads=NCPU)
    esc = _escapes_analytic(a, consts[2][sel], consts[3][sel], rp, 1000.0)
    assert set(np.unique(o["status"])) <= {KS.ST_CAPTURED, KS.ST_ESCAPED}
    wrong = (o["status"] == KS.ST_ESCAPED) != esc
    assert wrong.sum() == 0, (int(wrong.sum()), sel[wrong][:10])
    assert 0.2 < esc.mean() < 0.95
    he = o["health"][o["status"] == KS.ST_ESCAPED]
    assert np.median(he) < 1e-8 and he.max() < 1e-4        # the largest: rays that whirl ~2000 steps next to the photon orbit
    assert (o["steps_done"] + o["rejected"]).mean() < 1500          # per-ray step control: hundreds of attempts, not 10^5 steps
