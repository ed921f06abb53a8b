"""Pins of the oracle's RK4 loop, stop rules, events and snapshots (CPU only).

Pinned to: the paper's printed worked example, circular-orbit
closed forms (eqs.(27),(29),(40)), textbook photon orbits, exact constants of
motion, O(h^4) convergence (eqs.(41)-(43)), the analytic
capture/escape criterion for null rays (roots of the radial potential), and the
DESIGN.md readings B1-B6 / S1-S3 of the stop and snapshot semantics.
"""
import math
import os

import numpy as np
import pytest

from paper_1803_08320_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
PI2 = math.pi / 2


def _rows(name):
    out = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                out.append([float(x) for x in line.split()])
    return out


def _st(cols):
    return np.ascontiguousarray(np.array(cols, dtype=np.float64).T)


def test_worked_example_printed_digits(oracle):
    """PAPER.md:266-270 ICs, 278-316 output (tau t x y z), Schwarzschild h = 0.1.
    Cartesian via eq.(7) PAPER.md:88-93 typed here (a = 0)."""
    ics = _rows("ic_table.txt")[:2]
    st = _st([[r, 1.5708, 0.0, 0.0, 0.0, pph] for r, _, pph in ics])   # the 4-digit printed ICs
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, st, 0.1, 2, snapshot_every=1)
    snaps = res["snapshots"]                                            # [n][3][8]
    for part, tau, t, x, y, z in _rows("worked_example.txt"):
        i, k = int(part) - 1, int(round(tau / 0.1))
        s = snaps[i, k]
        r, th, ph = s[1], s[2], s[3]
        xyz = (r * math.sin(th) * math.cos(ph), r * math.sin(th) * math.sin(ph), r * math.cos(th))
        assert abs(s[0] - t) < 1.0e-4, (part, tau, s[0], t)
        for got, want in zip(xyz, (x, y, z)):
            assert abs(got - want) < 1.0e-4, (part, tau, xyz)


def test_schwarzschild_circular_orbits_closed_forms(oracle):
    """Config-1 shape.  r constant, phi = L tau / r^2 (eq.(40)),
    t = E tau/(1-2M/r) (eq.(29)), E = eq.(34), period T = 2 pi r^2/L."""
    st = W.circular_schwarzschild(64)
    h, n = 0.01, 2000
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, st, h, n, snapshot_every=100)
    f = res["final_state"]
    r0, L = st[0], st[5]
    tau = h * n
    assert np.max(np.abs(f[1] - r0)) < 1e-12              # r constant (p_r stays at rounding level)
    assert np.all(np.abs(f[5]) < 1e-13) and np.all(np.abs(f[6]) < 1e-13) and np.all(np.abs(f[2] - PI2) < 1e-13)
    E = (r0 - 2) / np.sqrt(r0 * (r0 - 3))
    assert np.allclose(f[4], E, rtol=1e-14)
    assert np.allclose(f[3], L * tau / r0 ** 2, rtol=1e-12)
    assert np.allclose(f[0], E * tau / (1 - 2 / r0), rtol=1e-12)
    assert np.all(res["status"] == oracle.ST_MAXSTEPS) and np.all(res["steps_done"] == n)
    assert np.all(res["snap_count"] == 21)
    assert np.all(res["health"] < 1e-13)
    # one full period returns phi = 2 pi
    r = 8.0
    Lc = r / math.sqrt(r - 3)
    T = 2 * math.pi * r * r / Lc
    nst = 4096
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[r, PI2, 0, 0, 0, Lc]]), T / nst, nst)
    assert abs(res["final_state"][3, 0] - 2 * math.pi) < 1e-11


def test_kerr_circular_orbit_frequency_eq27(oracle):
    """eq.(27) PAPER.md:190 with Table 1/2 rows moved outward to stable radii via BPT E, L."""
    for a, sgn in ((0.5, 1), (0.9, 1), (0.5, -1)):
        r = 10.0
        sa = sgn * a                                   # BPT closed forms (paper ref.[17]), M = 1
        den = r ** 0.75 * math.sqrt(r ** 1.5 - 3 * math.sqrt(r) + 2 * sa)
        E = (r ** 1.5 - 2 * math.sqrt(r) + sa) / den
        L = sgn * (r * r - 2 * sa * math.sqrt(r) + a * a) / den
        res = oracle.integrate(oracle.KERR, 1.0, a, _st([[r, PI2, 0, 0, 0, L]]), 0.01, 5000)
        f = res["final_state"][:, 0]
        assert abs(f[4] - E) < 1e-13
        assert abs(f[1] - r) < 1e-11 and abs(f[5]) < 1e-12
        D = 2 * r - a * a - r * r
        omega = (-2 * a * E + (2 - r) * L) / (r * D)   # eq.(27)
        assert abs(f[3] - omega * 50.0) < 1e-10
        assert abs(omega) == pytest.approx(1.0 / (r ** 1.5 + sa) * f[0] / 50.0, rel=1e-10)  # dphi/dt = 1/(r^1.5 +- a)


def test_photon_orbits(oracle):
    """Schwarzschild photon sphere r = 3M (lower limit of circular orbits) with
    L/E = 3 sqrt(3) M; Kerr equatorial photon orbits r_ph = 2M[1+cos(2/3 arccos(-+a/M))]
    (Bardeen-Press-Teukolsky).  Unstable: r stays for O(100) steps, then departs."""
    b = 3 * math.sqrt(3.0)
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[3.0, PI2, 0, 0, 0, b]]), 0.01, 200,
                           kind=oracle.NULL)
    f = res["final_state"][:, 0]
    assert abs(f[4] - 1.0) < 1e-15                       # E = 1 from the null mass shell
    assert abs(f[1] - 3.0) < 1e-9
    for a in (0.5, 0.9):
        for sgn in (1, -1):
            rph = 2 * (1 + math.cos(2.0 / 3.0 * math.acos(-sgn * a)))
            # impact parameter of the circular photon orbit: xi = -(r^3 - 3r^2 + a^2 r + a^2)/(a (r-1))
            xi = -(rph ** 3 - 3 * rph ** 2 + a * a * rph + a * a) / (a * (rph - 1))
            # scale so that E = 1: u_phi = xi
            res = oracle.integrate(oracle.KERR, 1.0, a, _st([[rph, PI2, 0, 0, 0, xi]]), 0.01, 100,
                                   kind=oracle.NULL)
            f = res["final_state"][:, 0]
            assert abs(f[4] - 1.0) < 1e-9, (a, sgn, f[4])
            assert abs(f[1] - rph) < 1e-6, (a, sgn, f[1], rph)
            assert (xi > 0) == (sgn > 0)


def _carter(a, f, kappa):
    th, E, pth, L = f[2], f[4], f[6], f[7]
    return pth ** 2 + np.cos(th) ** 2 * (a * a * (kappa - E * E) + L * L / np.sin(th) ** 2)


def test_constants_of_motion_and_h4_drift(oracle):
    """E, L_z exactly constant (eqs.(13)); 2H + kappa and Carter Q drift O(h^4)."""
    a = 0.9
    st, consts = W.kerr_bound(64, a, W.SEED_BASE + 2, return_constants=True)
    E0, L0, Q0 = consts
    drift = {}
    for h, n in ((0.1, 1000), (0.05, 2000)):
        res = oracle.integrate(oracle.KERR, 1.0, a, st, h, n)
        f = res["final_state"]
        assert np.array_equal(f[7], st[5])
        assert np.allclose(f[4], E0, rtol=1e-12)         # mass shell reproduces the drawn E
        Q = _carter(a, f, 1.0)
        drift[h] = (np.abs(Q - Q0), res["health"])
    dQ4, H4 = drift[0.1]
    dQ2, H2 = drift[0.05]
    big = dQ4 > 1e-9                                      # truncation-dominated particles only
    assert big.sum() >= 5
    ratio = np.median(dQ4[big] / dQ2[big])
    # O(h^4) bound; the secular part of an invariant's drift under RK4 is O(h^5) (e.g. the
    # harmonic oscillator: |R(i h w)|^2 = 1 - (h w)^6/72), so the ratio sits between 2^4 and 2^5.
    assert 12 < ratio < 40, ratio
    bigH = H4 > 1e-11
    assert bigH.sum() >= 5
    assert 12 < np.median(H4[bigH] / H2[bigH]) < 40
    assert np.max(H2) < 1e-6


def test_self_convergence_q16(oracle):
    """eqs.(41)-(43) PAPER.md:424-432: Q = |y_h - y_h/2| / |y_h/2 - y_h/4| -> 2^4 (Fig.8, 442)."""
    st = W.kerr_bound(10, 0.5, 99)
    sol = {}
    for h, n in ((0.2, 500), (0.1, 1000), (0.05, 2000)):
        sol[h] = oracle.integrate(oracle.KERR, 1.0, 0.5, st, h, n)["final_state"]
    num = np.linalg.norm(sol[0.2] - sol[0.1], axis=0)
    den = np.linalg.norm(sol[0.1] - sol[0.05], axis=0)
    q = num / den
    assert np.all(q > 11) and np.all(q < 24), q
    assert abs(np.median(q) - 16) < 2.5


def test_plain_and_compensated_updates_agree_and_long_double(oracle):
    """Reading P1: Kahan update is the same RK4; differences are rounding only."""
    st = W.kerr_bound(32, 0.9, 5)
    a = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.01, 20000)["final_state"]
    b = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.01, 20000, flags=oracle.FLAG_PLAIN_UPDATE)["final_state"]
    c = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.01, 20000, long_double=True)["final_state"]
    sc = np.maximum(np.abs(c), 1.0)
    assert np.max(np.abs(a - c) / sc) < 1e-10
    assert np.max(np.abs(b - c) / sc) < 1e-8
    assert np.max(np.abs(a - c) / sc) <= np.max(np.abs(b - c) / sc) * 1.5 + 1e-13


def _null_class_analytic(a, Lz, Q, r_plus, r_obs):
    """E = 1: R(r) = r^4 + (a^2 - L^2 - Q) r^2 + 2[Q + (L-a)^2] r - a^2 Q; an incoming ray escapes
    iff R has a real root (turning point) in (r_+, r_obs)."""
    out = np.zeros(Lz.size, dtype=bool)
    for i in range(Lz.size):
        roots = np.roots([1.0, 0.0, a * a - Lz[i] ** 2 - Q[i], 2 * (Q[i] + (Lz[i] - a) ** 2), -a * a * Q[i]])
        real = roots[np.abs(roots.imag) < 1e-9].real
        out[i] = np.any((real > r_plus) & (real < r_obs))
    return out


def test_null_camera_termination_class_matches_analytic_criterion(oracle):
    """Config-3 shape on a coarse 12x12 image: class == analytic turning-point criterion."""
    a = 0.998
    st, consts = W.camera_rays(12, a, 60.0, return_constants=True)
    al, be, Lz, Q = consts
    rp = W.horizon_radius(1.0, a)
    res = oracle.integrate(oracle.KERR, 1.0, a, st, 0.02, 200000, r_capture=rp + 0.01, r_escape=1100.0,
                           kind=oracle.NULL, nthreads=8)
    esc = _null_class_analytic(a, Lz, Q, rp, 1000.0)
    status = res["status"]
    assert np.all(np.isin(status, (oracle.ST_CAPTURED, oracle.ST_ESCAPED)))
    assert np.array_equal(status == oracle.ST_ESCAPED, esc)
    assert 0.05 < np.mean(~esc) < 0.4
    f = res["final_state"]
    assert np.all(f[1][esc] > 1100.0) and np.all(f[1][~esc] >= rp + 0.01)
    assert np.all(np.abs(f[4] - 1.0) < 1e-9)                  # photon normalisation E = 1 (reading N1)
    assert np.all(res["health"][esc] < 1e-6)                  # captured rays end in the BL-singular zone
    ec = res["eq_cross_r"]
    assert np.mean(np.isfinite(ec)) > 0.8 and np.nanmin(ec) > rp


def test_stop_rule_semantics(oracle):
    """Readings B1-B4."""
    L = 4.0
    # B1: y0 already inside the capture radius -> CAPTURED, 0 steps, final = y0
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[2.5, PI2, 0, 0, 0, L]]), 0.01, 10, r_capture=3.0)
    assert res["status"][0] == oracle.ST_CAPTURED and res["steps_done"][0] == 0
    assert res["final_state"][1, 0] == 2.5 and res["final_state"][0, 0] == 0.0
    # B1: already outside r_escape -> ESCAPED, 0 steps
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[50.0, PI2, 0, 0, 0, L]]), 0.01, 10, r_escape=40.0)
    assert res["status"][0] == oracle.ST_ESCAPED and res["steps_done"][0] == 0
    # B2: radial plunge; final state is the last accepted one (r >= r_capture), steps counted
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[6.0, PI2, 0, -0.5, 0, 0.0]]), 0.05, 100000,
                           r_capture=2.05)
    assert res["status"][0] == oracle.ST_CAPTURED
    assert res["final_state"][1, 0] >= 2.05 and res["final_state"][1, 0] < 2.2
    k = int(res["steps_done"][0])
    assert 0 < k < 100000
    again = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[6.0, PI2, 0, -0.5, 0, 0.0]]), 0.05, k)
    assert np.array_equal(again["final_state"], res["final_state"])     # exactly k accepted steps
    assert again["status"][0] == oracle.ST_MAXSTEPS
    # B3: outgoing photon escapes; final is the first post-step state beyond r_escape
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[10.0, PI2, 0, 1.2, 0, 2.0]]), 0.05, 100000,
                           r_escape=20.0, kind=oracle.NULL)
    assert res["status"][0] == oracle.ST_ESCAPED and res["final_state"][1, 0] > 20.0
    k = int(res["steps_done"][0])
    prev = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[10.0, PI2, 0, 1.2, 0, 2.0]]), 0.05, k - 1,
                            kind=oracle.NULL)
    assert prev["final_state"][1, 0] <= 20.0
    # nsteps = 0
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[10.0, PI2, 0, 0, 0, L]]), 0.05, 0)
    assert res["status"][0] == oracle.ST_MAXSTEPS and res["steps_done"][0] == 0
    # negative h integrates backwards: forward then backward returns to the start
    st = W.kerr_bound(4, 0.5, 3)
    fw = oracle.integrate(oracle.KERR, 1.0, 0.5, st, 0.01, 500)["final_state"]
    back_in = np.ascontiguousarray(fw[[1, 2, 3, 5, 6, 7]])
    bw = oracle.integrate(oracle.KERR, 1.0, 0.5, back_in, -0.01, 500)["final_state"]
    assert np.allclose(bw[[1, 2, 5, 6]], st[[0, 1, 3, 4]], rtol=0, atol=1e-9)


def test_equatorial_crossing_event(oracle):
    """Reading B5 on an orbit with known crossing: Schwarzschild circular orbit tilted out of the
    equatorial plane has r = const, so eq_cross_r must equal r to rounding."""
    r = 10.0
    Ltot = r / math.sqrt(r - 3)
    inc = 0.4                                            # orbital-plane tilt
    th0 = PI2 - 0.3
    # start at the top part of a tilted circle: L_z = Ltot cos(inc); p_theta from Q = Ltot^2 - L_z^2
    Lz = Ltot * math.cos(inc)
    pth2 = Ltot ** 2 - Lz ** 2 / math.sin(th0) ** 2
    assert pth2 > 0
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[r, th0, 0, 0, math.sqrt(pth2), Lz]]), 0.01, 3000)
    assert abs(res["eq_cross_r"][0] - r) < 1e-9
    assert abs(res["final_state"][1, 0] - r) < 1e-9
    # never crossing: equatorial orbit -> NaN
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[r, PI2, 0, 0, 0, Ltot]]), 0.01, 100)
    assert math.isnan(res["eq_cross_r"][0])


def test_snapshot_semantics(oracle):
    """Readings S1-S3: slot 0 = y0, slot j = state after j*every accepted steps (== final of a run
    with nsteps = j*every, bitwise), capacity respected, mask selects components."""
    st = W.kerr_bound(8, 0.9, 17)
    res = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.02, 1000, snapshot_every=250)
    assert res["snapshots"].shape == (8, 5, 8) and np.all(res["snap_count"] == 5)
    s = res["snapshots"]
    assert np.array_equal(s[:, 0, 1], st[0]) and np.all(s[:, 0, 0] == 0.0)
    assert np.array_equal(s[:, 0, 7], st[5]) and np.array_equal(s[:, 0, 5], st[3])
    for j in (1, 2, 4):
        part = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.02, 250 * j)["final_state"]
        assert np.array_equal(s[:, j, :].T, part)
    # capacity smaller than needed: extra slots dropped but counted
    res2 = oracle.integrate(oracle.KERR, 1.0, 0.9, st, 0.02, 1000, snapshot_every=250, snap_capacity=3,
                            snap_mask=0b00001110)
    assert res2["snapshots"].shape == (8, 3, 3) and np.all(res2["snap_count"] == 5)
    assert np.array_equal(res2["snapshots"], s[:, :3, 1:4])
    # nothing written after termination
    res3 = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, _st([[6.0, PI2, 0, -0.5, 0, 0.0]]), 0.05, 100000,
                            r_capture=2.05, snapshot_every=10)
    k = int(res3["steps_done"][0])
    assert res3["snap_count"][0] == 1 + k // 10
    assert np.all(np.isnan(res3["snapshots"][0, res3["snap_count"][0]:]))


def test_invalid_arguments(oracle):
    st = _st([[10.0, PI2, 0, 0, 0, 4.0]])
    with pytest.raises(ValueError):
        oracle.integrate(oracle.KERR, 1.0, 1.5, st, 0.01, 1)
    with pytest.raises(ValueError):
        oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.3, st, 0.01, 1)
    with pytest.raises(ValueError):
        oracle.integrate(oracle.KERR, 1.0, 0.5, st, 0.0, 1)


def test_cartesian_snapshots_are_the_papers_output_format(oracle):
    """snapshot records in the paper's output format (PAPER.md:318 'numerical solutions
    are stored in Cartesian coordinates'), eq.(7) PAPER.md:88-93.  Pins: the digits of the printed
    listing PAPER.md:278-316 (columns tau t x y z, reading G6) read straight from the oracle's records,
    and the oblate-spheroidal identity (x^2+y^2)/(r^2+a^2) + z^2/r^2 = 1 with tan(phi) = y/x in Kerr."""
    ics = _rows("ic_table.txt")[:2]
    st = _st([[r, 1.5708, 0.0, 0.0, 0.0, pph] for r, _, pph in ics])
    res = oracle.integrate(oracle.SCHWARZSCHILD, 1.0, 0.0, st, 0.1, 2, snapshot_every=1, snap_mask=0x0F,
                           flags=oracle.FLAG_CARTESIAN_SNAP)
    for part, tau, t, x, y, z in _rows("worked_example.txt"):
        rec = res["snapshots"][int(part) - 1, int(round(tau / 0.1))]          # (t, x, y, z)
        assert np.max(np.abs(rec - np.array([t, x, y, z]))) < 1.0e-4, (part, tau, rec)
    a = 0.9
    st = W.kerr_bound(40, a, W.SEED_BASE + 2)
    bl = oracle.integrate(oracle.KERR, 1.0, a, st, 0.01, 3000, snapshot_every=500)["snapshots"]
    ca = oracle.integrate(oracle.KERR, 1.0, a, st, 0.01, 3000, snapshot_every=500,
                          flags=oracle.FLAG_CARTESIAN_SNAP)["snapshots"]
    r, ph = bl[..., 1], bl[..., 3]
    x, y, z = ca[..., 1], ca[..., 2], ca[..., 3]
    assert np.max(np.abs((x * x + y * y) / (r * r + a * a) + z * z / (r * r) - 1.0)) < 1e-13
    assert np.max(np.abs(np.arctan2(y, x) - np.arctan2(np.sin(ph), np.cos(ph)))) < 1e-12
    for k in (0, 4, 5, 6, 7):                                              # the other components are untouched
        assert np.array_equal(bl[..., k], ca[..., k])
    assert np.all(np.sign(z) == np.sign(np.cos(bl[..., 2])))


def _scaled(st, M):
    """Geometrized units: lengths, times, L and p_theta scale with M; p_r, E, angles do not."""
    s = st.copy()
    s[0] *= M          # r
    s[4] *= M          # u_theta
    s[5] *= M          # u_phi = L
    return s


def test_mass_scaling_and_spin_reflection_symmetries(oracle):
    """Two exact symmetries of metric (6) that no implementation detail can fake:
    (i) M-scaling: the solution for (M, aM, h M) from scaled data is the M = 1 solution with lengths, t, L,
    p_theta multiplied by M; (ii) a -> -a together with L -> -L, phi -> -phi."""
    a, M = 0.7, 2.5
    st = W.kerr_bound(64, a, W.SEED_BASE + 2)
    r1 = oracle.integrate(oracle.KERR, 1.0, a, st, 0.01, 3000, r_capture=2.0, r_escape=100.0)
    rM = oracle.integrate(oracle.KERR, M, a * M, _scaled(st, M), 0.01 * M, 3000, r_capture=2.0 * M, r_escape=100.0 * M)
    scale = np.array([M, M, 1, 1, 1, 1, M, M])[:, None]            # t r th ph E pr pth L
    assert np.array_equal(r1["status"], rM["status"]) and np.array_equal(r1["steps_done"], rM["steps_done"])
    assert np.max(np.abs(rM["final_state"] / scale - r1["final_state"]) / np.maximum(np.abs(r1["final_state"]), 1)) < 1e-11
    flip = st.copy()
    flip[5] *= -1.0
    rf = oracle.integrate(oracle.KERR, 1.0, -a, flip, 0.01, 3000, r_capture=2.0, r_escape=100.0)
    sign = np.array([1, 1, 1, -1, 1, 1, 1, -1])[:, None]
    assert np.max(np.abs(rf["final_state"] * sign - r1["final_state"])) < 1e-11
