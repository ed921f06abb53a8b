"""Pins of the CPU oracle (oracle/geo_oracle.cpp) to what the paper and the
mathematics fix -- NOT to itself.  CPU only (``-m "not gpu"``).

Each test names the passage of /root/reference/PAPER.md (cited as PAPER.md:line)
or the textbook fact it pins to.  Formulas typed here are the PAPER's printed
equations (equatorial eqs.(9)-(12), Schwarzschild closed forms (34)-(40), metric
(6)); the oracle's Kerr RHS uses a different (separable) algebra, so agreement is
a real check.  The general (non-equatorial) Kerr RHS is pinned by high-precision
numerical differentiation of H = 1/2 g^{mu nu} p_mu p_nu with g^{mu nu} obtained
by numerically inverting the printed metric (6) -- no derivative formula shared.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

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


# ---------------------------------------------------------------------------
# metric (6), typed from the paper; H by numerical inversion
# ---------------------------------------------------------------------------
def _metric6(M, a, r, th):
    s, c = mp.sin(th), mp.cos(th)
    rho2 = r * r + a * a * c * c
    Delta = r * r - 2 * M * r + a * a
    Sigma = (r * r + a * a) ** 2 - a * a * Delta * s * s
    g = mp.zeros(4, 4)                          # order t, r, theta, phi
    g[0, 0] = -(1 - 2 * M * r / rho2)
    g[0, 3] = g[3, 0] = -2 * M * a * r * s * s / rho2
    g[1, 1] = rho2 / Delta
    g[2, 2] = rho2
    g[3, 3] = Sigma * s * s / rho2
    return g


def _H_mp(M, a, r, th, pt_std, pr, pth, pph):
    ginv = mp.inverse(_metric6(M, a, r, th))
    p = mp.matrix([pt_std, pr, pth, pph])
    return (p.T * ginv * p)[0] / 2


def _rhs_by_differentiation(M, a, y8):
    """Hamilton's equations (3),(4) PAPER.md:60-65 by mp.diff of H; p_t(std) = -E (reading G1)."""
    mp.mp.dps = 40
    t, r, th, ph, E, pr, pth, L = [mp.mpf(float(v)) for v in y8]
    M, a = mp.mpf(M), mp.mpf(a)
    pt = -E
    dt = mp.diff(lambda x: _H_mp(M, a, r, th, x, pr, pth, L), pt)
    dr = mp.diff(lambda x: _H_mp(M, a, r, th, pt, x, pth, L), pr)
    dth = mp.diff(lambda x: _H_mp(M, a, r, th, pt, pr, x, L), pth)
    dph = mp.diff(lambda x: _H_mp(M, a, r, th, pt, pr, pth, x), L)
    dpr = -mp.diff(lambda x: _H_mp(M, a, x, th, pt, pr, pth, L), r)
    dpth = -mp.diff(lambda x: _H_mp(M, a, r, x, pt, pr, pth, L), th)
    return np.array([float(v) for v in (dt, dr, dth, dph, dpr, dpth)])


def _close(x, y, rel):
    return abs(x - y) <= rel * max(abs(y), 1.0)


@pytest.mark.parametrize("a", [0.0, 0.5, 0.9, 0.998])
def test_kerr_rhs_matches_numerical_hamilton_equations(oracle, a):
    """Full (non-equatorial) RHS == dH/dp, -dH/dx of metric (6)."""
    rng = np.random.default_rng(7)
    for _ in range(6):
        r = rng.uniform(2.2, 30.0)
        th = rng.uniform(0.3, math.pi - 0.3)
        y = [0.0, r, th, rng.uniform(0, 6), rng.uniform(0.9, 1.1), rng.uniform(-0.3, 0.3),
             rng.uniform(-2, 2), rng.uniform(-4, 4)]
        want = _rhs_by_differentiation(1.0, a, y)
        got = oracle.rhs(oracle.KERR, 1.0, a, y)
        for g, w in zip(got, want):
            assert _close(g, w, 2e-13), (a, y, got, want)


def test_kerr_rhs_matches_paper_equatorial_eqs_9_to_12(oracle):
    """eqs.(9)-(12), typed as printed (p_t = E, reading G1)."""
    rng = np.random.default_rng(11)
    for _ in range(20):
        M = 1.0
        a = rng.uniform(0.0, 0.998)
        r = rng.uniform(2.5, 25.0)
        pt, pr, pph = rng.uniform(0.8, 1.2), rng.uniform(-0.5, 0.5), rng.uniform(-4, 4)
        D = 2 * M * r - a * a - r * r
        tdot = (-(2 * M * a * a + a * a * r + r ** 3) * pt + 2 * a * M * pph) / (r * D)       # (9)
        rdot = -D / r ** 2 * pr                                                             # (10)
        phdot = (-2 * M * a * pt + (2 * M - r) * pph) / (r * D)                              # (11)
        prdot = (-(M * r - a * a) / r ** 3 * pr ** 2                                         # (12)
                 + M * (4 * M * a * a * r - a ** 4 - 2 * a * a * r * r - r ** 4) / (r * r * D * D) * pt ** 2
                 - 2 * M * a * (4 * M * r - a * a - 3 * r * r) / (r * r * D * D) * pt * pph
                 + (4 * M * M * r - M * a * a - 4 * M * r * r + r ** 3) / (r * r * D * D) * pph ** 2)
        d = oracle.rhs(oracle.KERR, M, a, [0, r, PI2, 0.3, pt, pr, 0.0, pph])
        assert _close(d[0], tdot, 1e-13) and _close(d[1], rdot, 1e-13)
        assert _close(d[3], phdot, 1e-13) and _close(d[4], prdot, 1e-13)
        assert d[2] == 0.0 and abs(d[5]) < 1e-15                                            # (13)


def test_schwarzschild_rhs_is_a_to_zero_limit_and_hamiltonian(oracle):
    """eqs.(29)-(32) PAPER.md:203-211 (oracle's Schwarzschild branch, typed from the paper)
    == Kerr branch at a=0 == numerical Hamilton equations of metric (6) at a=0."""
    rng = np.random.default_rng(3)
    for _ in range(8):
        y = [0.0, rng.uniform(2.5, 30), rng.uniform(0.2, 2.9), 1.0, rng.uniform(0.9, 1.1),
             rng.uniform(-0.4, 0.4), rng.uniform(-3, 3), rng.uniform(-4, 4)]
        ds = oracle.rhs(oracle.SCHWARZSCHILD, 1.0, 0.0, y)
        dk = oracle.rhs(oracle.KERR, 1.0, 0.0, y)
        dn = _rhs_by_differentiation(1.0, 0.0, y)
        for s_, k_, n_ in zip(ds, dk, dn):
            assert _close(s_, k_, 5e-14) and _close(s_, n_, 5e-14)


def test_long_double_rhs_agrees(oracle):
    y = [0.0, 5.3, 1.1, 0.2, 0.95, 0.1, 1.3, 2.2]
    d = oracle.rhs(oracle.KERR, 1.0, 0.9, y)
    dl = oracle.rhs(oracle.KERR, 1.0, 0.9, y, long_double=True)
    assert np.allclose(d, dl, rtol=1e-14, atol=1e-15)


# ---------------------------------------------------------------------------
# mass shell (eq.(5)): printed E values
# ---------------------------------------------------------------------------
def test_energy_matches_printed_ic_table(oracle):
    """PAPER.md:268-270 rows (r, p_t, p_phi), 4 digits; L from eq.(35)/(39) exactly."""
    for r, pt, pph in _rows("ic_table.txt"):
        L = r / math.sqrt(r - 3.0)                                   # eq.(39), M = 1
        assert abs(L - pph) < 6e-5
        E = oracle.energy(1.0, 0.0, r, PI2, 0.0, 0.0, L, 1.0)
        assert abs(E - pt) < 6e-5
        assert abs(E - math.sqrt((r - 2) ** 2 / (r * (r - 3)))) < 1e-14   # eq.(34)


def test_energy_and_circularity_match_isco_tables(oracle):
    """Tables 1-2 PAPER.md:385-416 (13 digits): with (r, p_phi) printed, the mass shell must
    give the printed p_t, and p_r-dot must vanish (circular orbit, eq.(14)).
    ISCO = marginal stability: d(p_r-dot)/dr = 0 there (eq.(20))."""
    for sense, a, r, pt, pph in _rows("isco_tables.txt"):
        if a == 1.0 and sense > 0:
            continue            # r = r_+ = M: BL coordinates singular (PAPER.md:174 takes a limit)
        E = oracle.energy(1.0, a, r, PI2, 0.0, 0.0, pph, 1.0)
        assert abs(E - pt) < 2e-11, (sense, a, E, pt)
        f = lambda rr: oracle.rhs(oracle.KERR, 1.0, a, [0, rr, PI2, 0, pt, 0.0, 0.0, pph])[4]
        assert abs(f(r)) < 5e-12
        eps = 1e-4
        slope = (f(r + eps) - f(r - eps)) / (2 * eps)
        assert abs(slope) < 1e-8, (sense, a, slope)


def test_extreme_kerr_retrograde_isco_closed_form(oracle):
    """eq.(23): r=9M, L=-22M/(3 sqrt 3), E=5/(3 sqrt 3)."""
    L = -22.0 / (3 * math.sqrt(3))
    E = oracle.energy(1.0, 1.0, 9.0, PI2, 0.0, 0.0, L, 1.0)
    assert abs(E - 5.0 / (3 * math.sqrt(3))) < 1e-14
    assert abs(oracle.rhs(oracle.KERR, 1.0, 1.0, [0, 9.0, PI2, 0, E, 0, 0, L])[4]) < 1e-15


def test_hamiltonian_is_mass_shell(oracle):
    rng = np.random.default_rng(5)
    for kappa in (0.0, 1.0):
        for _ in range(10):
            r, th = rng.uniform(2.5, 40), rng.uniform(0.3, 2.8)
            pr, pth, L = rng.uniform(-.3, .3), rng.uniform(-2, 2), rng.uniform(-4, 4)
            E = oracle.energy(1.0, 0.7, r, th, pr, pth, L, kappa)
            assert E > 0
            twoH = 2 * oracle.hamiltonian(1.0, 0.7, [0, r, th, 0, E, pr, pth, L])
            assert abs(twoH + kappa) < 1e-12
            mp.mp.dps = 30
            assert abs(float(2 * _H_mp(1, mp.mpf(0.7), mp.mpf(r), mp.mpf(th), -mp.mpf(E), mp.mpf(pr),
                                       mp.mpf(pth), mp.mpf(L))) + kappa) < 1e-12
