"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path
(tests, bench).  It holds none of the method's arithmetic: no RHS, no RK4, no
mass-shell solve, no stop rule.  It only draws constants of motion / positions
and turns them into the ``state_in`` SoA ``[6][n] = (r, theta, phi, u_r,
u_theta, u_phi)`` that ``geo_integrate`` (include/geo.h) and
``oracle_integrate`` (oracle/geo_oracle.cpp) both take.

The paper's own initial conditions are unpublished "random" sets
(PAPER.md:436, 446 -- sec. 6.3, 6.4); these recipes stand in for them
(DESIGN.md "Input recipe").  All in geometrized units G=c=1.

PRNG: counter-based SplitMix64-style mixer, uniform = top 53 bits * 2^-53.
Draw ``k`` of stream ``seed`` is ``mix(seed + (k+1)*GOLDEN)``; candidate ``j``
of a rejection sampler consumes draws ``7j .. 7j+6`` and candidates are accepted
in candidate order, so the output does not depend on the chunk size.
"""
from __future__ import annotations

import math
import numpy as np

SEED_BASE = 180308320          # config k uses seed SEED_BASE + k
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix_uniform(seed: int, idx: np.ndarray) -> np.ndarray:
    """Uniform doubles in [0,1) for draw indices ``idx`` (any int array) of stream ``seed``."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (idx.astype(np.uint64) + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# ----------------------------------------------------------------------------
# closed forms used only to SHAPE the inputs
# ----------------------------------------------------------------------------
def horizon_radius(M: float, a: float) -> float:
    """r_+ = M + sqrt(M^2 - a^2)."""
    return M + math.sqrt(M * M - a * a)


def bpt_isco(M: float, a: float, prograde: bool = True) -> float:
    """ISCO radius, Bardeen-Press-Teukolsky Z1/Z2 form (paper ref. [17]; the
    reading G4 of eq.(21), agrees with it -- tests pin both to
    Tables 1-2)."""
    x = a / M
    z1 = 1.0 + (1.0 - x * x) ** (1.0 / 3.0) * ((1.0 + x) ** (1.0 / 3.0) + (1.0 - x) ** (1.0 / 3.0))
    z2 = math.sqrt(3.0 * x * x + z1 * z1)
    s = -1.0 if prograde else 1.0
    return M * (3.0 + z2 + s * math.sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2)))


def circular_schwarzschild(n: int, seed: int = SEED_BASE + 1, M: float = 1.0,
                           r_lo: float = 6.5, r_hi: float = 20.0) -> np.ndarray:
    """Config 1: equatorial circular timelike orbits, r ~ U[r_lo, r_hi]*M.
    u_phi = L from eq.(35) PAPER.md:222 (L^2 = M r^2/(r-3M)); theta = pi/2,
    phi = 0, u_r = u_theta = 0 (eqs.(14),(33) PAPER.md:120, 217).  p_t is NOT an
    input: the method derives it from eq.(5)."""
    u = splitmix_uniform(seed, np.arange(n))
    r = (r_lo + (r_hi - r_lo) * u) * M
    st = np.zeros((6, n), dtype=np.float64)
    st[0] = r
    st[1] = math.pi / 2
    st[5] = r * np.sqrt(M / (r - 3.0 * M))
    return st


def _carter_R_coeffs(E, Lz, Q, M, a):
    """Coefficients (c4..c0) of the timelike radial potential
    R(r) = [E(r^2+a^2) - a Lz]^2 - Delta [r^2 + (Lz - aE)^2 + Q]."""
    e1 = E * E - 1.0
    c4 = e1
    c3 = 2.0 * M + 0.0 * E
    c2 = a * a * e1 - Lz * Lz - Q
    c1 = 2.0 * M * ((Lz - a * E) ** 2 + Q)
    c0 = -a * a * Q
    return c4, c3, c2, c1, c0


def _poly4(c4, c3, c2, c1, c0, r):
    return (((c4 * r + c3) * r + c2) * r + c1) * r + c0


def _cubic_real_roots(A, B, C, D):
    """Real roots of A x^3 + B x^2 + C x + D (A != 0), vectorised.  Returns an
    array [3][m]; missing roots are NaN."""
    b = B / A
    c = C / A
    d = D / A
    p = c - b * b / 3.0
    q = 2.0 * b ** 3 / 27.0 - b * c / 3.0 + d
    disc = (q / 2.0) ** 2 + (p / 3.0) ** 3
    out = np.full((3,) + A.shape, np.nan)
    three = disc <= 0.0
    # three real roots (trigonometric form)
    with np.errstate(invalid="ignore", divide="ignore"):
        m = 2.0 * np.sqrt(np.maximum(-p / 3.0, 0.0))
        arg = np.where(m > 0, 3.0 * q / (p * m), 0.0)
        ang = np.arccos(np.clip(arg, -1.0, 1.0)) / 3.0
        for k in range(3):
            out[k] = np.where(three, m * np.cos(ang - 2.0 * math.pi * k / 3.0) - b / 3.0, np.nan)
        # one real root (Cardano)
        sq = np.sqrt(np.maximum(disc, 0.0))
        one = np.cbrt(-q / 2.0 + sq) + np.cbrt(-q / 2.0 - sq) - b / 3.0
        out[0] = np.where(three, out[0], one)
    return out


def kerr_bound(n: int, a: float, seed: int, M: float = 1.0, r_hi: float = 30.0,
               chunk: int = 1 << 21, return_constants: bool = False, nthreads: int = 1):
    """Configs 2 / 4 (reading W1): bound, non-plunging timelike Kerr orbits.

    Candidate j draws (r0, theta0, E, Lz, Q, sgn_r, sgn_theta) with
    r0 ~ U[1.2 r_isco(prograde, a), r_hi M], theta0 ~ U[pi/6, 5pi/6],
    E ~ U[0.90, 0.98], Lz ~ U[-4, 4] M, Q ~ U[0, 12] M^2, signs +-1.
    Accept iff Theta(theta0) >= 0, R(r0) >= 0 and R is negative somewhere in
    (r_+, r0) -- i.e. an inner turning point exists outside the horizon (E < 1
    already bounds the orbit from above).  Because R(r_+) >= 0 always, that is
    the case iff some critical point of R inside (r_+, r0) has R < 0.
    Then u_r = sgn_r sqrt(R)/Delta, u_theta = sgn_theta sqrt(Theta), u_phi = Lz,
    phi0 = 0.
    """
    r_lo = 1.2 * bpt_isco(M, a, True)
    r_p = horizon_radius(M, a)

    def one_chunk(j0):
        j = np.arange(j0, j0 + chunk, dtype=np.int64)
        d = [splitmix_uniform(seed, 7 * j + k) for k in range(7)]
        r0 = r_lo + (r_hi * M - r_lo) * d[0]
        th0 = math.pi / 6 + (2 * math.pi / 3) * d[1]
        E = 0.90 + 0.08 * d[2]
        Lz = (-4.0 + 8.0 * d[3]) * M
        Q = 12.0 * d[4] * M * M
        sr = np.where(d[5] < 0.5, -1.0, 1.0)
        sth = np.where(d[6] < 0.5, -1.0, 1.0)
        s2 = np.sin(th0) ** 2
        c2 = np.cos(th0) ** 2
        Theta = Q - c2 * (a * a * (1.0 - E * E) + Lz * Lz / s2)
        c4, c3, c2_, c1, c0 = _carter_R_coeffs(E, Lz, Q, M, a)
        R0 = _poly4(c4, c3, c2_, c1, c0, r0)
        ok = (Theta >= 0.0) & (R0 >= 0.0)
        idx = np.nonzero(ok)[0]
        if idx.size:
            cr = _cubic_real_roots(4.0 * c4[idx], 3.0 * c3[idx], 2.0 * c2_[idx], c1[idx])
            neg = np.zeros(idx.size, dtype=bool)
            for k in range(3):
                x = cr[k]
                with np.errstate(invalid="ignore"):
                    inside = (x > r_p) & (x < r0[idx])
                    val = _poly4(c4[idx], c3[idx], c2_[idx], c1[idx], c0[idx], np.where(inside, x, 1.0))
                    neg |= inside & (val < 0.0)
            idx = idx[neg]
        r = r0[idx]
        Delta = r * r - 2.0 * M * r + a * a
        st = np.zeros((6, idx.size))
        st[0] = r
        st[1] = th0[idx]
        st[3] = sr[idx] * np.sqrt(R0[idx]) / Delta
        st[4] = sth[idx] * np.sqrt(Theta[idx])
        st[5] = Lz[idx]
        return st, np.stack([E[idx], Lz[idx], Q[idx]])

    cols = []
    consts = []
    have = 0
    j0 = 0
    pool = None
    if nthreads > 1:
        from concurrent.futures import ThreadPoolExecutor
        pool = ThreadPoolExecutor(nthreads)
    try:
        while have < n:
            # chunks are taken in candidate order, so the result does not depend on nthreads
            starts = [j0 + k * chunk for k in range(max(1, nthreads))]
            j0 += chunk * len(starts)
            results = list(pool.map(one_chunk, starts)) if pool else [one_chunk(starts[0])]
            for st, cs in results:
                cols.append(st)
                consts.append(cs)
                have += st.shape[1]
    finally:
        if pool:
            pool.shutdown()
    st = np.ascontiguousarray(np.concatenate(cols, axis=1)[:, :n])
    if return_constants:
        return st, np.ascontiguousarray(np.concatenate(consts, axis=1)[:, :n])
    return st


def camera_rays(N: int, a: float, incl_deg: float, M: float = 1.0, r_obs: float = 1000.0,
                width: float = 20.0, row0: int = 0, rows: int | None = None,
                return_constants: bool = False):
    """Configs 3 / 5 (reading N2): Bardeen image plane at finite r_obs, one photon
    per pixel, E = 1.  Pixel (ix, iy): alpha = (ix + 1/2 - N/2) W/N,
    beta = (iy + 1/2 - N/2) W/N, particle index (iy-row0)*N + ix.
    Lz = -alpha sin i, Q = beta^2 + (alpha^2 - a^2) cos^2 i; start
    (r, theta, phi) = (r_obs, i, 0); u_r = -sqrt(max(R,0))/Delta with
    R = [(r^2+a^2) - a Lz]^2 - Delta[(Lz-a)^2 + Q]; u_theta = -beta; u_phi = Lz.
    ``row0, rows`` select a horizontal tile (config 5 is tiled, reading S3).
    No randomness: the image is the seed."""
    if rows is None:
        rows = N - row0
    inc = math.radians(incl_deg)
    si, ci = math.sin(inc), math.cos(inc)
    ix = np.arange(N, dtype=np.float64)
    iy = np.arange(row0, row0 + rows, dtype=np.float64)
    al = ((ix + 0.5 - N / 2) * (width * M / N))[None, :].repeat(rows, 0).ravel()
    be = ((iy + 0.5 - N / 2) * (width * M / N))[:, None].repeat(N, 1).ravel()
    Lz = -al * si
    Q = be * be + (al * al - a * a) * ci * ci
    r = r_obs * M
    Delta = r * r - 2.0 * M * r + a * a
    R = ((r * r + a * a) - a * Lz) ** 2 - Delta * ((Lz - a) ** 2 + Q)
    n = al.size
    st = np.zeros((6, n))
    st[0] = r
    st[1] = inc
    st[3] = -np.sqrt(np.maximum(R, 0.0)) / Delta
    st[4] = -be
    st[5] = Lz
    if return_constants:
        return st, np.stack([al, be, Lz, Q])
    return st


# ----------------------------------------------------------------------------
# Tabulated 3+1 metrics: input DATA for geo_create_tabulated / oracle_tab_integrate --
# the five functions of eq.(8) sampled on a uniform (x^1, x^2) grid.  No interpolation, no
# equations of motion here.
# ----------------------------------------------------------------------------
def kerr_metric_table(M: float, a: float, n1: int, n2: int, x1_lo: float, x1_hi: float,
                      x2_lo: float = 0.0, x2_hi: float = math.pi, radial: str = "r", ghost: int = 2) -> dict:
    """alpha, beta^phi, gamma_11, gamma_22, gamma_33 of the Kerr metric, eq.(8), at the nodes of a
    uniform grid: ``n1 x n2`` nodes span [x1_lo, x1_hi] x [x2_lo, x2_hi] and ``ghost`` more nodes are added on every
    side (the cubic-convolution stencil needs one; eq.(8) is analytic there, also beyond theta = 0, pi).
    radial = "r": x^1 = r (Boyer-Lindquist);  radial = "log": x^1 = ln(r - r_+), r = r_+ + exp(x^1), so that
    gamma_11 = gamma_rr (dr/dx^1)^2 = rho^2 (r - r_+)/(r - r_-) is regular at the horizon and a uniform grid
    resolves both the near-horizon region and the far field.  Returns {"tab": [5][n2+2g][n1+2g], "x1_0", "d1",
    "x2_0", "d2"} (x1_0, x2_0: coordinates of node 0, ghosts included)."""
    d1 = (x1_hi - x1_lo) / (n1 - 1)
    d2 = (x2_hi - x2_lo) / (n2 - 1)
    x1 = x1_lo + d1 * (np.arange(n1 + 2 * ghost) - ghost)
    x2 = x2_lo + d2 * (np.arange(n2 + 2 * ghost) - ghost)
    X1, TH = np.meshgrid(x1, x2)                       # [n2][n1], x^1 fastest
    rp, rm = M + math.sqrt(M * M - a * a), M - math.sqrt(M * M - a * a)
    if radial == "log":
        ex = np.exp(X1)
        r = rp + ex
        jac2_over_delta = ex / (r - rm)                # (dr/dx1)^2 / Delta = (r - r_+)^2 / ((r - r_+)(r - r_-))
    elif radial == "r":
        r = X1
        jac2_over_delta = 1.0 / (r * r - 2.0 * M * r + a * a)
    else:
        raise ValueError(radial)
    s2 = np.sin(TH) ** 2
    rho2 = r * r + a * a * np.cos(TH) ** 2
    Delta = r * r - 2.0 * M * r + a * a
    Sigma = (r * r + a * a) ** 2 - a * a * Delta * s2
    tab = np.empty((5,) + r.shape)
    tab[0] = np.sqrt(rho2 * Delta / Sigma)
    tab[1] = -2.0 * M * a * r / Sigma
    tab[2] = rho2 * jac2_over_delta
    tab[3] = rho2
    tab[4] = Sigma / rho2 * s2
    return {"tab": np.ascontiguousarray(tab), "x1_0": float(x1[0]), "d1": float(d1), "x2_0": float(x2[0]), "d2": float(d2),
            "radial": radial, "r_plus": rp}


def general_table_from_diagonal(table: dict) -> dict:
    """The ten-field layout of a GENERAL stationary axisymmetric 3+1 metric (reading T6: alpha, beta^1, beta^2,
    beta^3, gamma_11, gamma_12, gamma_13, gamma_22, gamma_23, gamma_33) holding a five-field table of eq.(8)'s structure
    (beta^1 = beta^2 = 0, diagonal gamma_ij): the same metric in the wider layout."""
    t5 = table["tab"]
    z = np.zeros_like(t5[0])
    out = dict(table)
    out["tab"] = np.ascontiguousarray(np.stack([t5[0], z, z, t5[1], t5[2], z, z, t5[3], z, t5[4]]))
    return out


def kerr_schild_metric_table(M: float, a: float, n1: int, n2: int, r_lo: float, r_hi: float,
                             x2_lo: float = 0.0, x2_hi: float = math.pi, ghost: int = 2) -> dict:
    """Input data for reading T6: the Kerr metric in ingoing Kerr-Schild (horizon-penetrating) coordinates
    (t~, r, theta, phi~), dt~ = dt + 2Mr/Delta dr, dphi~ = dphi + a/Delta dr, whose line element
        ds^2 = -(1 - f) dt~^2 + 2 f dt~ dr - 2 a f s^2 dt~ dphi~ + (1 + f) dr^2 + rho^2 dtheta^2
               - 2 a (1 + f) s^2 dr dphi~ + (r^2 + a^2 + a^2 f s^2) s^2 dphi~^2,     f = 2 M r / rho^2,  s = sin theta,
    is regular at r = r_+.  Its 3+1 split (line element (1)): gamma_ij = g_ij, beta_i = g_ti,
    beta^i = gamma^{ij} beta_j, alpha^2 = beta_i beta^i - g_tt -- here beta^r = f/(1 + f) != 0 and gamma_r phi != 0, i.e. a
    metric OUTSIDE the structure of eq.(8).  Nodes and ghosts as in kerr_metric_table; no interpolation, no equations of
    motion here."""
    d1 = (r_hi - r_lo) / (n1 - 1)
    d2 = (x2_hi - x2_lo) / (n2 - 1)
    x1 = r_lo + d1 * (np.arange(n1 + 2 * ghost) - ghost)
    x2 = x2_lo + d2 * (np.arange(n2 + 2 * ghost) - ghost)
    r, TH = np.meshgrid(x1, x2)
    s2 = np.sin(TH) ** 2
    rho2 = r * r + a * a * np.cos(TH) ** 2
    f = 2.0 * M * r / rho2
    g = np.zeros(r.shape + (3, 3))
    g[..., 0, 0] = 1.0 + f
    g[..., 1, 1] = rho2
    g[..., 2, 2] = (r * r + a * a + a * a * f * s2) * s2
    g[..., 0, 2] = g[..., 2, 0] = -a * (1.0 + f) * s2
    bl = np.stack([f, np.zeros_like(f), -a * f * s2], axis=-1)           # beta_i = g_ti
    bu = np.linalg.solve(g, bl[..., None])[..., 0]                       # beta^i
    alpha = np.sqrt((bl * bu).sum(-1) + (1.0 - f))
    tab = np.stack([alpha, bu[..., 0], bu[..., 1], bu[..., 2], g[..., 0, 0], g[..., 0, 1], g[..., 0, 2], g[..., 1, 1],
                    g[..., 1, 2], g[..., 2, 2]])
    return {"tab": np.ascontiguousarray(tab), "x1_0": float(x1[0]), "d1": float(d1), "x2_0": float(x2[0]), "d2": float(d2),
            "r_plus": M + math.sqrt(M * M - a * a)}


def to_kerr_schild(st: np.ndarray, E: np.ndarray, M: float, a: float) -> np.ndarray:
    """state_in (r, theta, phi, u_r, u_theta, u_phi) of Boyer-Lindquist data with energy E -> the same covector in ingoing
    Kerr-Schild coordinates: p_r~ = p_r + (2 M r E - a L)/Delta (from p_mu dx^mu invariant, p_t = -E); r, theta, p_theta,
    p_phi unchanged; phi~ = phi at the start (the coordinate offset is a constant of the transformation)."""
    out = np.array(st, dtype=np.float64, copy=True)
    r = st[0]
    Delta = r * r - 2.0 * M * r + a * a
    out[3] = st[3] + (2.0 * M * r * E - a * st[5]) / Delta
    return out


def to_cartesian_kerr_schild(st: np.ndarray, E: np.ndarray, M: float, a: float) -> np.ndarray:
    """state_in (r, theta, phi, u_r, u_theta, u_phi) of Boyer-Lindquist data with energy E -> the same event and covector in
    CARTESIAN Kerr-Schild coordinates, state_in (x, y, z, p_x, p_y, p_z) of a GEO_KERR_SCHILD ctx (reading K1):
    first `to_kerr_schild` (ingoing Kerr coordinates, phi~ = phi at the start), then the point transformation
        x + i y = (r + i a) sin(theta) exp(i phi~),   z = r cos(theta),
    whose Jacobian J[i][b] = d x^i / d(r, theta, phi~)^b carries the covector: p_b = J[i][b] p_i, solved for p_i (3 x 3
    per particle; needs sin(theta) != 0 -- the spherical chart, not the Cartesian one, is singular on the axis).
    A change of coordinates of the input data; no equations of motion here."""
    ks = to_kerr_schild(st, E, M, a)
    r, th, ph = ks[0], ks[1], ks[2]
    s, c = np.sin(th), np.cos(th)
    sp, cp = np.sin(ph), np.cos(ph)
    x = (r * cp - a * sp) * s
    y = (r * sp + a * cp) * s
    z = r * c
    J = np.zeros((st.shape[1], 3, 3))
    J[:, 0, 0] = cp * s
    J[:, 0, 1] = (r * cp - a * sp) * c
    J[:, 0, 2] = -y
    J[:, 1, 0] = sp * s
    J[:, 1, 1] = (r * sp + a * cp) * c
    J[:, 1, 2] = x
    J[:, 2, 0] = c
    J[:, 2, 1] = -r * s
    J[:, 2, 2] = 0.0
    p_sph = np.stack([ks[3], ks[4], ks[5]], axis=-1)
    p_cart = np.linalg.solve(np.transpose(J, (0, 2, 1)), p_sph[..., None])[..., 0]
    return np.ascontiguousarray(np.stack([x, y, z, p_cart[:, 0], p_cart[:, 1], p_cart[:, 2]]))


def kerr_schild_radius(xyz: np.ndarray, a: float) -> np.ndarray:
    """Kerr-Schild radius r(x, y, z): the non-negative root of r^4 - (x^2 + y^2 + z^2 - a^2) r^2 - a^2 z^2 = 0; xyz [3][n].
    Used by tests and the bench to compare a Cartesian Kerr-Schild result with a Boyer-Lindquist one (the charts share r
    and cos(theta) = z / r)."""
    x, y, z = xyz[0], xyz[1], xyz[2]
    w = x * x + y * y + z * z - a * a
    return np.sqrt(0.5 * (w + np.sqrt(w * w + 4.0 * a * a * z * z)))


def to_log_radial(st: np.ndarray, r_plus: float) -> np.ndarray:
    """state_in (r, theta, phi, u_r, u_theta, u_phi) -> the same covectors in x^1 = ln(r - r_+): u_1 = u_r (r - r_+)."""
    out = np.array(st, dtype=np.float64, copy=True)
    out[0] = np.log(st[0] - r_plus)
    out[3] = st[3] * (st[0] - r_plus)
    return out


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous particle-index range [lo, hi) of ``rank`` (geodesics
    are independent, PAPER.md:329 -- no exchange step)."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def interleaved_tiles(ntiles: int, rank: int, world: int) -> list[int]:
    """Image tiles of ``rank``: tile t -> rank t mod world, so every rank gets the same
    captured/escaped mix (captured rays cost about half an escaping one)."""
    return list(range(rank, ntiles, world))
