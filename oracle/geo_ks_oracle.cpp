// geo_ks_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow CPU oracle for SURVEY 8(f).3, second clause ("further analytic metrics / horizon-penetrating,
// axis-regular coordinates", the paper's motivation for the 3+1 form): fixed-step classical RK4
// of independent null / timelike geodesics of the Kerr metric (6) written in CARTESIAN
// KERR-SCHILD coordinates (t~, x, y, z) -- DESIGN.md readings K1-K5.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline leg may build, load or call this file.  It shares no code with the CUDA path.
//
// The metric (Kerr 1963; Kerr & Schild 1965), ingoing form, G = c = 1:
//     g_{mu nu} = eta_{mu nu} + f l_mu l_nu,          eta = diag(-1, 1, 1, 1),
//     f   = 2 M r^3 / (r^4 + a^2 z^2),
//     l_mu = ( 1, (r x + a y)/(r^2 + a^2), (r y - a x)/(r^2 + a^2), z / r ),
//     r(x, y, z) >= 0 the root of   (x^2 + y^2)/(r^2 + a^2) + z^2 / r^2 = 1
//                  <=>  r^4 - (x^2 + y^2 + z^2 - a^2) r^2 - a^2 z^2 = 0.
// l is null for eta and for g, hence g^{mu nu} = eta^{mu nu} - f l^mu l^nu with l^mu = eta^{mu nu} l_nu = (-1, l_x, l_y, l_z).
// It is metric (6) of the paper under  t~ = t + int 2Mr/Delta dr,  phi~ = phi + int a/Delta dr,
// x + i y = (r + i a) sin(theta) exp(i phi~),  z = r cos(theta)   (tests/test_oracle_ks.py pulls the matrix back through the
// Jacobian of this map and compares with eq.(6) entry by entry).  3+1 split, line element (1) PAPER.md:47:
//     alpha^2 = 1/(1 + f),   beta^i = f l_i / (1 + f),   gamma_ij = delta_ij + f l_i l_j.
//
// Equations of motion: Hamilton's equations (3),(4) of H = 1/2 g^{mu nu} p_mu p_nu.  With the paper's
// sign p_t(paper) = E = -p_t (reading G1) and  lP = l^mu p_mu = E + l_j p_j:
//     H        = 1/2 [ -E^2 + p_x^2 + p_y^2 + p_z^2 - f lP^2 ]
//     dt~/dtau = dH/dp_t = E + f lP
//     dx^i/dtau = dH/dp_i = p_i - f lP l_i
//     dp_i/dtau = -dH/dx^i = 1/2 (d_i f) lP^2 + f lP sum_j p_j d_i l_j
//     dE/dtau = 0 (the metric does not depend on t~).
// Every partial derivative below is written out by the quotient rule, one line per entry, in the order of the formulas
// above; no collected terms, no reciprocals shared.  The pins (tests/test_oracle_ks.py) are: the pull-back to eq.(6); finite
// differences of H from the numerically inverted 4 x 4 matrix in 40-digit arithmetic; the 3+1 identities; the mass shell;
// geodesics of the pinned Boyer-Lindquist oracle transformed into this chart (r, cos(theta) = z/r, E, L_z = x p_y - y p_x and
// Carter's constant agree at common tau); exact straight lines at M = 0; conservation of L_z, Q, 2H across the polar axis
// and through the horizon, where the Boyer-Lindquist oracle cannot go.
//
// RK4, the Kahan update (reading P1), the stop rules and the record semantics are those of geo_oracle.cpp
// (readings B1-B6, S1-S3) with r := r(x, y, z) and the equatorial plane z = 0 (readings K2, K3).
//
// Build: with geo_oracle.cpp into libgeo_oracle.so (oracle/build.py), -O2 -ffp-contract=off.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <limits>
#include <thread>
#include <vector>

#include "dp45.h"

namespace {

enum { KS_ST_MAXSTEPS = 0, KS_ST_CAPTURED = 1, KS_ST_ESCAPED = 2, KS_ST_NUMERIC = 3 };
enum { KS_FLAG_PLAIN_UPDATE = 1 };

template <class R> struct KsHole { R M, a; };

// State in the paper's order with the chart's own coordinates: (t~, x, y, z, p_t = E, p_x, p_y, p_z).
template <class R> struct KsState { R t, x, y, z, E, px, py, pz; };

// d/dtau of (t~, x, y, z, p_x, p_y, p_z)
template <class R> struct KsDeriv { R t, x, y, z, px, py, pz; };

// r(x, y, z): the non-negative root of r^4 - w r^2 - a^2 z^2 = 0, w = x^2 + y^2 + z^2 - a^2.
template <class R> R ks_radius(const KsHole<R>& bh, R x, R y, R z) {
    const R a = bh.a;
    const R w = x * x + y * y + z * z - a * a;
    const R disc = std::sqrt(w * w + R(4) * a * a * z * z);
    return std::sqrt((w + disc) / R(2));
}

// f, l_mu and their gradients at one point, all by the quotient rule.
template <class R> struct KsGeom {
    R r, f, l[3];     // l[0..2] = l_x, l_y, l_z
    R dr[3];          // d_i r
    R df[3];          // d_i f
    R dl[3][3];       // dl[i][j] = d_i l_j
};

template <class R> KsGeom<R> ks_geometry(const KsHole<R>& bh, R x, R y, R z) {
    const R M = bh.M, a = bh.a;
    KsGeom<R> g;
    const R r = ks_radius(bh, x, y, z);
    g.r = r;
    const R r2 = r * r, r3 = r2 * r, r4 = r2 * r2;
    const R S = r4 + a * a * z * z;          // denominator of f
    const R A = r2 + a * a;                  // denominator of l_x, l_y
    g.f = R(2) * M * r3 / S;
    g.l[0] = (r * x + a * y) / A;
    g.l[1] = (r * y - a * x) / A;
    g.l[2] = z / r;
    // implicit differentiation of F(r; x, y, z) = r^4 - w r^2 - a^2 z^2 = 0:  d_i r = -(dF/dx_i) / (dF/dr)
    const R w = x * x + y * y + z * z - a * a;
    const R Fr = R(4) * r3 - R(2) * w * r;
    g.dr[0] = R(2) * x * r2 / Fr;
    g.dr[1] = R(2) * y * r2 / Fr;
    g.dr[2] = (R(2) * z * r2 + R(2) * a * a * z) / Fr;
    for (int i = 0; i < 3; ++i) {
        const R dS = R(4) * r3 * g.dr[i] + (i == 2 ? R(2) * a * a * z : R(0));
        const R dA = R(2) * r * g.dr[i];
        g.df[i] = R(2) * M * (R(3) * r2 * g.dr[i] * S - r3 * dS) / (S * S);
        // numerators of l_x, l_y:  N_x = r x + a y,  N_y = r y - a x
        const R dNx = g.dr[i] * x + (i == 0 ? r : R(0)) + (i == 1 ? a : R(0));
        const R dNy = g.dr[i] * y + (i == 1 ? r : R(0)) - (i == 0 ? a : R(0));
        g.dl[i][0] = (dNx * A - (r * x + a * y) * dA) / (A * A);
        g.dl[i][1] = (dNy * A - (r * y - a * x) * dA) / (A * A);
        g.dl[i][2] = ((i == 2 ? R(1) : R(0)) * r - z * g.dr[i]) / r2;
    }
    return g;
}

// H = 1/2 g^{mu nu} p_mu p_nu = 1/2 [ -E^2 + p^2 - f (E + l.p)^2 ]            (eq.(4))
template <class R> R ks_hamiltonian(const KsHole<R>& bh, const KsState<R>& y) {
    const KsGeom<R> g = ks_geometry(bh, y.x, y.y, y.z);
    const R lP = y.E + g.l[0] * y.px + g.l[1] * y.py + g.l[2] * y.pz;
    return (-y.E * y.E + y.px * y.px + y.py * y.py + y.pz * y.pz - g.f * lP * lP) / R(2);
}

// Hamilton's equations (3)
template <class R> KsDeriv<R> ks_rhs(const KsHole<R>& bh, const KsState<R>& y) {
    const KsGeom<R> g = ks_geometry(bh, y.x, y.y, y.z);
    const R p[3] = {y.px, y.py, y.pz};
    const R lP = y.E + g.l[0] * p[0] + g.l[1] * p[1] + g.l[2] * p[2];
    KsDeriv<R> d;
    d.t = y.E + g.f * lP;
    d.x = p[0] - g.f * lP * g.l[0];
    d.y = p[1] - g.f * lP * g.l[1];
    d.z = p[2] - g.f * lP * g.l[2];
    R dp[3];
    for (int i = 0; i < 3; ++i) {
        const R pdl = p[0] * g.dl[i][0] + p[1] * g.dl[i][1] + p[2] * g.dl[i][2];
        dp[i] = g.df[i] * lP * lP / R(2) + g.f * lP * pdl;
    }
    d.px = dp[0]; d.py = dp[1]; d.pz = dp[2];
    return d;
}

// Mass shell eq.(5) PAPER.md:69 in the 3+1 variables of line element (1): E = alpha sqrt(kappa + gamma^{ij} p_i p_j) - beta^k p_k
// with alpha^2 = 1/(1+f), beta^i = f l_i/(1+f), gamma^{ij} = delta^{ij} - f l_i l_j/(1+f)   (future-directed root).
template <class R> R ks_energy(const KsHole<R>& bh, R x, R y, R z, R px, R py, R pz, R kappa) {
    const KsGeom<R> g = ks_geometry(bh, x, y, z);
    const R lp = g.l[0] * px + g.l[1] * py + g.l[2] * pz;
    const R alpha = R(1) / std::sqrt(R(1) + g.f);
    const R gpp = px * px + py * py + pz * pz - g.f * lp * lp / (R(1) + g.f);
    const R betap = g.f * lp / (R(1) + g.f);
    return alpha * std::sqrt(kappa + gpp) - betap;
}

struct KsStop { double r_capture, r_escape; int32_t kind; int32_t flags; };

struct KsOut {
    double* final_state;    // [8][n]  t~, x, y, z, E, p_x, p_y, p_z
    int32_t* status;
    int64_t* steps_done;
    double* eq_cross_r;     // [n] or null: r at the first crossing of z = 0 (reading K3)
    double* health;         // [n] or null: |2H + kappa|
    double* snapshots;      // [n][snap_capacity][ncomp] or null
    int64_t snap_capacity;
    uint32_t snap_mask;
    int32_t* snap_count;
};

template <class R> R ks_component(const KsState<R>& y, int k) {
    switch (k) {
        case 0: return y.t;  case 1: return y.x;  case 2: return y.y;  case 3: return y.z;
        case 4: return y.E;  case 5: return y.px; case 6: return y.py; default: return y.pz;
    }
}

template <class R> bool ks_finite7(const KsState<R>& y) {
    return std::isfinite(y.t) && std::isfinite(y.x) && std::isfinite(y.y) && std::isfinite(y.z) &&
           std::isfinite(y.px) && std::isfinite(y.py) && std::isfinite(y.pz);
}

template <class R> KsState<R> ks_shifted(const KsState<R>& y, R w, const KsDeriv<R>& k) {
    KsState<R> s = y;
    s.t = y.t + w * k.t;
    s.x = y.x + w * k.x;
    s.y = y.y + w * k.y;
    s.z = y.z + w * k.z;
    s.px = y.px + w * k.px;
    s.py = y.py + w * k.py;
    s.pz = y.pz + w * k.pz;
    return s;
}

template <class R> void ks_kahan_add(R& y, R& c, R delta, bool plain) {
    if (plain) { y = y + delta; return; }
    const R yk = delta - c;
    const R tsum = y + yk;
    c = (tsum - y) - yk;
    y = tsum;
}

template <class R> void ks_write_snapshot(const KsOut& o, int64_t i, int64_t slot, const KsState<R>& y) {
    if (!o.snapshots || slot >= o.snap_capacity) return;   // S3
    int ncomp = 0;
    for (int k = 0; k < 8; ++k) ncomp += (o.snap_mask >> k) & 1u;
    double* dst = o.snapshots + (i * o.snap_capacity + slot) * ncomp;
    int j = 0;
    for (int k = 0; k < 8; ++k)
        if ((o.snap_mask >> k) & 1u) dst[j++] = (double)ks_component(y, k);
}

template <class R>
void ks_integrate_one(const KsHole<R>& bh, const double* state_in, int64_t n, int64_t i, R h, int64_t nsteps,
                      const KsStop& st, int64_t snapshot_every, const KsOut& o) {
    const R kappa = st.kind == 0 ? R(1) : R(0);
    const bool plain = (st.flags & KS_FLAG_PLAIN_UPDATE) != 0;
    const R rc = (R)st.r_capture, re = (R)st.r_escape;

    KsState<R> y;
    y.t = R(0);
    y.x = (R)state_in[0 * n + i];
    y.y = (R)state_in[1 * n + i];
    y.z = (R)state_in[2 * n + i];
    y.px = (R)state_in[3 * n + i];
    y.py = (R)state_in[4 * n + i];
    y.pz = (R)state_in[5 * n + i];
    y.E = ks_energy(bh, y.x, y.y, y.z, y.px, y.py, y.pz, kappa);
    R c[7] = {0, 0, 0, 0, 0, 0, 0};   // Kahan error terms of (t, x, y, z, px, py, pz)

    int32_t status = -1;
    int64_t steps = 0, snaps = 0;
    R eq_cross = std::numeric_limits<R>::quiet_NaN();
    bool crossed = false;
    R ry = ks_radius(bh, y.x, y.y, y.z);      // r of the current accepted state

    // B1 with r = r(x, y, z) (reading K2)
    if (!(ry >= rc)) status = KS_ST_CAPTURED;
    else if (!ks_finite7(y) || !std::isfinite(y.E)) status = KS_ST_NUMERIC;
    else {
        if (snapshot_every > 0) { ks_write_snapshot(o, i, 0, y); snaps = 1; }
        if (ry > re) status = KS_ST_ESCAPED;
        else if (nsteps == 0) status = KS_ST_MAXSTEPS;
    }

    while (status < 0) {
        // classical RK4; B2: capture guard on every evaluation point
        const KsDeriv<R> k1 = ks_rhs(bh, y);
        const KsState<R> y2 = ks_shifted(y, h / R(2), k1);
        if (!(ks_radius(bh, y2.x, y2.y, y2.z) >= rc)) { status = KS_ST_CAPTURED; break; }
        const KsDeriv<R> k2 = ks_rhs(bh, y2);
        const KsState<R> y3 = ks_shifted(y, h / R(2), k2);
        if (!(ks_radius(bh, y3.x, y3.y, y3.z) >= rc)) { status = KS_ST_CAPTURED; break; }
        const KsDeriv<R> k3 = ks_rhs(bh, y3);
        const KsState<R> y4 = ks_shifted(y, h, k3);
        if (!(ks_radius(bh, y4.x, y4.y, y4.z) >= rc)) { status = KS_ST_CAPTURED; break; }
        const KsDeriv<R> k4 = ks_rhs(bh, y4);

        KsState<R> yn = y;
        R cn[7] = {c[0], c[1], c[2], c[3], c[4], c[5], c[6]};
        const R w = h / R(6);
        ks_kahan_add(yn.t, cn[0], w * (k1.t + R(2) * k2.t + R(2) * k3.t + k4.t), plain);
        ks_kahan_add(yn.x, cn[1], w * (k1.x + R(2) * k2.x + R(2) * k3.x + k4.x), plain);
        ks_kahan_add(yn.y, cn[2], w * (k1.y + R(2) * k2.y + R(2) * k3.y + k4.y), plain);
        ks_kahan_add(yn.z, cn[3], w * (k1.z + R(2) * k2.z + R(2) * k3.z + k4.z), plain);
        ks_kahan_add(yn.px, cn[4], w * (k1.px + R(2) * k2.px + R(2) * k3.px + k4.px), plain);
        ks_kahan_add(yn.py, cn[5], w * (k1.py + R(2) * k2.py + R(2) * k3.py + k4.py), plain);
        ks_kahan_add(yn.pz, cn[6], w * (k1.pz + R(2) * k2.pz + R(2) * k3.pz + k4.pz), plain);

        const R rn = ks_radius(bh, yn.x, yn.y, yn.z);
        if (!(rn >= rc)) { status = KS_ST_CAPTURED; break; }        // B2: end point
        if (!ks_finite7(yn)) { status = KS_ST_NUMERIC; break; }     // B6

        if (!crossed) {                                             // reading K3: first sign change of z
            if (y.z * yn.z < R(0)) {
                crossed = true;
                eq_cross = ry + (rn - ry) * (R(0) - y.z) / (yn.z - y.z);
            }
        }
        y = yn;
        ry = rn;
        for (int k = 0; k < 7; ++k) c[k] = cn[k];
        ++steps;
        if (snapshot_every > 0 && steps % snapshot_every == 0) {    // S1
            ks_write_snapshot(o, i, snaps, y);
            ++snaps;
        }
        if (ry > re) status = KS_ST_ESCAPED;                        // B3
        else if (steps >= nsteps) status = KS_ST_MAXSTEPS;          // B4
    }

    for (int k = 0; k < 8; ++k) o.final_state[(int64_t)k * n + i] = (double)ks_component(y, k);
    o.status[i] = status;
    o.steps_done[i] = steps;
    if (o.eq_cross_r) o.eq_cross_r[i] = (double)eq_cross;
    if (o.health) o.health[i] = (double)std::fabs(R(2) * ks_hamiltonian(bh, y) + kappa);
    if (o.snap_count) o.snap_count[i] = (int32_t)snaps;
}

template <class R>
void ks_integrate_range(double M, double a, const double* state_in, int64_t n, int64_t lo, int64_t hi, double h,
                        int64_t nsteps, const KsStop& st, int64_t snapshot_every, const KsOut& o) {
    KsHole<R> bh{(R)M, (R)a};
    for (int64_t i = lo; i < hi; ++i) ks_integrate_one<R>(bh, state_in, n, i, (R)h, nsteps, st, snapshot_every, o);
}

// ---------------------------------------------------------------------------------------------------------------
// Reading K6: the adaptive Dormand-Prince 5(4) stepper of readings A1-A3 (geo_oracle.cpp: integrate_one_adaptive, the
// same pair, controller, landing rule and continuous extension, dp45.h) in this chart: the SEVEN evolving components
// (t~, x, y, z, p_x, p_y, p_z) enter the error norm.  Two rules differ from A2, both because far from the hole the
// geodesics of this chart are straight lines (the error estimate vanishes and the controller would grow h without bound):
//   K6a  step cap: no attempt moves the particle by more than a quarter of its current radius in coordinate distance,
//        h <- min(h, r / (4 |dx/dtau|)) with dx/dtau = k_1 (not in fixed-step mode, rtol = +inf) -- a step cannot jump
//        over (or into) the hole from afar without an evaluation point ever feeling it;
//   K6b  the capture test runs on y0 and on the END POINT of an attempt (r(x, y, z) < r_capture: CAPTURED, the attempt is
//        not taken), not on the stage points: the chart is regular through the horizon, a stage point inside the capture
//        radius is an ordinary evaluation point (in Cartesian components the stage points of a step along a tight orbit
//        cut the chord and dip below the orbit's radius by r (dphi)^2 / 8: with a guard on them, rays that skim the
//        prograde photon orbit 0.001 M outside the capture radius would be captured spuriously).
// Escape after an accepted step, event K3, records K5 at tau_j = j snap_dtau.
// ---------------------------------------------------------------------------------------------------------------
template <class R> R ks_comp7(const KsState<R>& y, int c) {
    switch (c) { case 0: return y.t; case 1: return y.x; case 2: return y.y; case 3: return y.z;
                 case 4: return y.px; case 5: return y.py; default: return y.pz; }
}
template <class R> R ks_dcomp7(const KsDeriv<R>& k, int c) {
    switch (c) { case 0: return k.t; case 1: return k.x; case 2: return k.y; case 3: return k.z;
                 case 4: return k.px; case 5: return k.py; default: return k.pz; }
}
template <class R> void ks_set7(KsState<R>& y, int c, R v) {
    switch (c) { case 0: y.t = v; break; case 1: y.x = v; break; case 2: y.y = v; break; case 3: y.z = v; break;
                 case 4: y.px = v; break; case 5: y.py = v; break; default: y.pz = v; }
}

template <class R>
void ks_integrate_one_adaptive(const KsHole<R>& bh, const double* state_in, int64_t n, int64_t i, const AdaptiveCtl& ctl,
                               int64_t max_attempts, const KsStop& st, const KsOut& o, int64_t* rejected_out) {
    static const DP45 T;
    const R kappa = st.kind == 0 ? R(1) : R(0);
    const R rc = (R)st.r_capture, re = (R)st.r_escape;
    KsState<R> y;
    y.t = R(0);
    y.x = (R)state_in[0 * n + i];
    y.y = (R)state_in[1 * n + i];
    y.z = (R)state_in[2 * n + i];
    y.px = (R)state_in[3 * n + i];
    y.py = (R)state_in[4 * n + i];
    y.pz = (R)state_in[5 * n + i];
    y.E = ks_energy(bh, y.x, y.y, y.z, y.px, y.py, y.pz, kappa);
    R cc[7] = {0, 0, 0, 0, 0, 0, 0};
    R h = (R)ctl.h0, tau = R(0);
    const R tau_end = (R)ctl.tau_end;
    const bool dense = ctl.snap_dtau > 0.0 && o.snapshots != nullptr;
    const R dtau = (R)ctl.snap_dtau;
    int64_t next_j = 0;
    int32_t status = -1;
    int64_t steps = 0, attempts = 0, rejected = 0;
    R eq_cross = std::numeric_limits<R>::quiet_NaN();
    bool crossed = false;
    R ry = ks_radius(bh, y.x, y.y, y.z);

    if (!(ry >= rc)) status = KS_ST_CAPTURED;                        // B1 / K2
    else if (!ks_finite7(y) || !std::isfinite(y.E)) status = KS_ST_NUMERIC;
    else {
        if (dense) { ks_write_snapshot(o, i, 0, y); next_j = 1; }
        if (ry > re) status = KS_ST_ESCAPED;
        else if (max_attempts == 0) status = KS_ST_MAXSTEPS;
    }

    KsDeriv<R> k[DP45::S];
    if (status < 0) k[0] = ks_rhs(bh, y);
    while (status < 0) {
        if (!std::isinf(ctl.rtol)) {                                 // K6a
            const R hcap = ry / (R(4) * std::sqrt(k[0].x * k[0].x + k[0].y * k[0].y + k[0].z * k[0].z));
            if (h > hcap) h = hcap;
        }
        const bool last = tau + R(1.01) * h >= tau_end;
        if (last) h = tau_end - tau;
        for (int s = 1; s < DP45::S - 1; ++s) {                      // stages 2..6 (no capture guard on them: K6b)
            KsState<R> ys = y;
            for (int c = 0; c < 7; ++c) {
                R acc = R(0);
                for (int j = 0; j < s; ++j) acc += (R)T.a[s][j] * ks_dcomp7(k[j], c);
                ks_set7(ys, c, ks_comp7(y, c) + h * acc);
            }
            k[s] = ks_rhs(bh, ys);
        }
        ++attempts;
        KsState<R> yn = y;
        R cn[7];
        for (int c = 0; c < 7; ++c) {
            R acc5 = R(0);
            for (int j = 0; j < DP45::S - 1; ++j) acc5 += (R)T.a[6][j] * ks_dcomp7(k[j], c);
            R v = ks_comp7(y, c);
            cn[c] = cc[c];
            ks_kahan_add(v, cn[c], h * acc5, false);
            ks_set7(yn, c, v);
        }
        const R rn = ks_radius(bh, yn.x, yn.y, yn.z);
        if (!(rn >= rc)) { status = KS_ST_CAPTURED; break; }         // end point
        const bool fin = ks_finite7(yn);
        R err = std::numeric_limits<R>::quiet_NaN();                 // a non-finite attempt: rejected, the step shrinks by 0.2
        if (fin) {
            err = R(0);
            k[6] = ks_rhs(bh, yn);
            for (int c = 0; c < 7; ++c) {
                R acce = R(0);
                for (int j = 0; j < DP45::S; ++j)
                    acce += ((R)(j < 6 ? T.a[6][j] : 0.0L) - (R)T.b4[j]) * ks_dcomp7(k[j], c);
                const R sc = (R)ctl.atol + (R)ctl.rtol * std::max(std::fabs(ks_comp7(y, c)), std::fabs(ks_comp7(yn, c)));
                const R ec = std::fabs(h * acce) / sc;
                if (!(ec <= err)) err = ec;
            }
        }
        if (fin && std::isinf(ctl.rtol)) err = R(0);
        R fac = err > R(0) ? R(0.9) * std::pow(err, R(-0.2)) : (err == R(0) ? R(5) : R(0.2));
        if (!(fac >= R(0.2))) fac = R(0.2);
        if (fac > R(5)) fac = R(5);
        if (std::isinf(ctl.rtol)) fac = R(1);
        if (!fin || !(err <= R(1))) {                                // reject
            ++rejected;
            h *= std::min(fac, R(1));
            if ((std::isinf(ctl.rtol) && !fin) || !(std::fabs(h) >= (R)ctl.h_min) || !(std::fabs(h) > R(0))) { status = KS_ST_NUMERIC; break; }
            if (attempts >= max_attempts) { status = KS_ST_MAXSTEPS; break; }
            continue;
        }
        if (!crossed && y.z * yn.z < R(0)) {                         // K3
            crossed = true;
            eq_cross = ry + (rn - ry) * (R(0) - y.z) / (yn.z - y.z);
        }
        const R tau_new = last ? tau_end : tau + h;
        if (dense) {
            for (;;) {
                const R tj = (R)next_j * dtau;
                if (!(tj <= tau_new)) break;
                R w[7];
                dp45_dense_weights<R>((tj - tau) / h, w);
                KsState<R> ys = y;
                for (int c = 0; c < 7; ++c) {
                    R acc = R(0);
                    for (int j = 0; j < DP45::S; ++j) acc += w[j] * ks_dcomp7(k[j], c);
                    ks_set7(ys, c, ks_comp7(y, c) + h * acc);
                }
                ks_write_snapshot(o, i, next_j, ys);
                ++next_j;
            }
        }
        y = yn;
        ry = rn;
        for (int c = 0; c < 7; ++c) cc[c] = cn[c];
        k[0] = k[6];
        ++steps;
        tau = tau_new;
        h *= fac;
        if (ry > re) status = KS_ST_ESCAPED;
        else if (last || attempts >= max_attempts) status = KS_ST_MAXSTEPS;
    }
    for (int q = 0; q < 8; ++q) o.final_state[(int64_t)q * n + i] = (double)ks_component(y, q);
    o.status[i] = status;
    o.steps_done[i] = steps;
    if (o.eq_cross_r) o.eq_cross_r[i] = (double)eq_cross;
    if (o.health) o.health[i] = (double)std::fabs(R(2) * ks_hamiltonian(bh, y) + kappa);
    if (dense && o.snap_count) o.snap_count[i] = (int32_t)next_j;
    if (rejected_out) rejected_out[i] = rejected;
}

}  // namespace

extern "C" {

// Returns 0 on success, 1 on invalid arguments.  HOST memory.  precision: 0 = double, 1 = long double.
// state_in [6][n] = (x, y, z, p_x, p_y, p_z).
int oracle_ks_integrate(double M, double a, const double* state_in, int64_t n, double h, int64_t nsteps,
                        const KsStop* stop, int64_t snapshot_every, const KsOut* out, int precision, int nthreads) {
    if (!stop || !out || n < 0 || nsteps < 0 || snapshot_every < 0) return 1;
    if (!(M >= 0) || !(std::fabs(a) <= M || M == 0) || !std::isfinite(h) || h == 0.0) return 1;
    if (n == 0) return 0;
    if (!state_in || !out->final_state || !out->status || !out->steps_done) return 1;
    if (snapshot_every > 0 && (!out->snapshots || !out->snap_count || out->snap_capacity < 1 ||
                               (out->snap_mask & 0xFFu) == 0)) return 1;
    if (nthreads < 1) nthreads = 1;
    if ((int64_t)nthreads > n) nthreads = (int)n;
    auto run = [&](int64_t lo, int64_t hi) {
        if (precision == 1) ks_integrate_range<long double>(M, a, state_in, n, lo, hi, h, nsteps, *stop, snapshot_every, *out);
        else ks_integrate_range<double>(M, a, state_in, n, lo, hi, h, nsteps, *stop, snapshot_every, *out);
    };
    if (nthreads == 1) { run(0, n); return 0; }
    std::vector<std::thread> pool;
    const int64_t block = 64;
    const int64_t nblocks = (n + block - 1) / block;
    for (int t = 0; t < nthreads; ++t)
        pool.emplace_back([&, t]() {
            for (int64_t b = t; b < nblocks; b += nthreads) run(b * block, std::min<int64_t>(n, (b + 1) * block));
        });
    for (auto& th : pool) th.join();
    return 0;
}

// d/dtau of (t~, x, y, z, p_x, p_y, p_z) at y8 = (t~, x, y, z, E, p_x, p_y, p_z)
void oracle_ks_rhs(double M, double a, const double* y8, double* d7, int precision) {
    if (precision == 1) {
        KsHole<long double> bh{M, a};
        KsState<long double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
        const KsDeriv<long double> d = ks_rhs(bh, y);
        d7[0] = (double)d.t; d7[1] = (double)d.x; d7[2] = (double)d.y; d7[3] = (double)d.z;
        d7[4] = (double)d.px; d7[5] = (double)d.py; d7[6] = (double)d.pz;
    } else {
        KsHole<double> bh{M, a};
        KsState<double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
        const KsDeriv<double> d = ks_rhs(bh, y);
        d7[0] = d.t; d7[1] = d.x; d7[2] = d.y; d7[3] = d.z; d7[4] = d.px; d7[5] = d.py; d7[6] = d.pz;
    }
}

double oracle_ks_hamiltonian(double M, double a, const double* y8) {
    KsHole<double> bh{M, a};
    KsState<double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
    return ks_hamiltonian(bh, y);
}

double oracle_ks_energy(double M, double a, double x, double y, double z, double px, double py, double pz, double kappa) {
    KsHole<double> bh{M, a};
    return ks_energy(bh, x, y, z, px, py, pz, kappa);
}

double oracle_ks_radius(double M, double a, double x, double y, double z) {
    KsHole<double> bh{M, a};
    return ks_radius(bh, x, y, z);
}

// f, l_x, l_y, l_z at a point (for the pull-back and 3+1 pins): out4 = (f, l_x, l_y, l_z)
void oracle_ks_metric(double M, double a, double x, double y, double z, double* out4) {
    KsHole<double> bh{M, a};
    const KsGeom<double> g = ks_geometry(bh, x, y, z);
    out4[0] = g.f; out4[1] = g.l[0]; out4[2] = g.l[1]; out4[3] = g.l[2];
}

// Adaptive RK5(4) in the Kerr-Schild chart (reading K6).  ctl = {h0, rtol, atol, h_min, tau_end, snap_dtau}; rejected: [n] or NULL.
int oracle_ks_integrate_adaptive(double M, double a, const double* state_in, int64_t n, const AdaptiveCtl* ctl,
                                 int64_t max_attempts, const KsStop* stop, const KsOut* out, int64_t* rejected,
                                 int precision, int nthreads) {
    if (!stop || !out || !ctl || n < 0 || max_attempts < 0) return 1;
    if (!(M >= 0) || !(std::fabs(a) <= M || M == 0)) return 1;
    if (!std::isfinite(ctl->h0) || !(ctl->h0 > 0.0) || !(ctl->rtol >= 0) || !(ctl->atol >= 0) || !(ctl->rtol + ctl->atol > 0) ||
        !(ctl->h_min >= 0) || !(ctl->tau_end > 0) || !(ctl->snap_dtau >= 0)) return 1;
    if (n == 0) return 0;
    if (!state_in || !out->final_state || !out->status || !out->steps_done) return 1;
    if (ctl->snap_dtau > 0 && (!out->snapshots || !out->snap_count || out->snap_capacity < 1 || (out->snap_mask & 0xFFu) == 0)) return 1;
    if (nthreads < 1) nthreads = 1;
    std::vector<std::thread> pool;
    const int64_t block = 64, nblocks = (n + block - 1) / block;
    for (int t = 0; t < nthreads; ++t)
        pool.emplace_back([&, t]() {
            for (int64_t b = t; b < nblocks; b += nthreads)
                for (int64_t i = b * block; i < std::min<int64_t>(n, (b + 1) * block); ++i) {
                    if (precision == 1) {
                        KsHole<long double> bh{M, a};
                        ks_integrate_one_adaptive<long double>(bh, state_in, n, i, *ctl, max_attempts, *stop, *out, rejected);
                    } else {
                        KsHole<double> bh{M, a};
                        ks_integrate_one_adaptive<double>(bh, state_in, n, i, *ctl, max_attempts, *stop, *out, rejected);
                    }
                }
        });
    for (auto& th : pool) th.join();
    return 0;
}

}  // extern "C"
