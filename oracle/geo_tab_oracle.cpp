// geo_tab_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, one-particle-at-a-time CPU oracle for SURVEY 8(f).3: fixed-step classical RK4 geodesics
// in a NUMERICALLY GIVEN (tabulated) stationary, axisymmetric 3+1 metric -- the "numerical metrics" the
// paper names as the reason for its 3+1 formulation.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or call
// this file.  It shares NO code with the CUDA path (paper_1803_08320_b200/csrc/).
//
// What it computes (readings T1-T5):
//   T1  Line element (1) with the structure of eq.(8): shift beta^i = (0,0,beta^phi),
//       gamma_ij = diag(gamma_11, gamma_22, gamma_33), all five functions of (x^1, x^2) only.  They are given at
//       the nodes x^1_i = x1_0 + i d1 (i < n1), x^2_j = x2_0 + j d2 (j < n2):  tab[f][j][i], f = 0..4 in the
//       order alpha, beta^phi, gamma_11, gamma_22, gamma_33.  (x^1, x^2) are the metric's own coordinates;
//       for Kerr in Boyer-Lindquist coordinates they are (r, theta).
//   T2  Between the nodes every field is the tensor-product CUBIC CONVOLUTION interpolant (Keys 1981,
//       parameter -1/2, "Catmull-Rom"): C^1, exact for polynomials of degree <= 2, third-order accurate.
//       With u = (x - x_0)/d, i = floor(u), s = u - i the four weights of the nodes i-1 .. i+2 are
//           w_-1 = (-s^3 + 2 s^2 - s)/2   w_0 = (3 s^3 - 5 s^2 + 2)/2   w_1 = (-3 s^3 + 4 s^2 + s)/2   w_2 = (s^3 - s^2)/2.
//       The derivatives in the equations of motion are the EXACT derivatives of that interpolant
//       (d/dx = (1/d) d/ds of the weights), so the system integrated is the Hamiltonian system (3),(4)
//        of the interpolated metric: p_t and p_phi are constants of motion exactly.
//   T3  Hamilton's equations of H = 1/2 [ -(p_t - beta^phi p_phi)^2/alpha^2 + p_1^2/gamma_11 + p_2^2/gamma_22
//       + p_phi^2/gamma_33 ]  (eq.(4) with the inverse of metric (1)), p_t = -E, p_phi = L, W = E + beta^phi L,
//       u^t = W/alpha^2:
//           dt/dtau = u^t,  dx^k/dtau = p_k/gamma_kk (k = 1, 2),  dphi/dtau = L/gamma_33 - beta^phi u^t,
//           dp_k/dtau = u^t L d_k beta^phi - alpha (u^t)^2 d_k alpha
//                       + 1/2 [ d_k gamma_11 (p_1/gamma_11)^2 + d_k gamma_22 (p_2/gamma_22)^2 + d_k gamma_33 (L/gamma_33)^2 ].
//       E from the mass shell (5): E = alpha sqrt(kappa + p_1^2/gamma_11 + p_2^2/gamma_22 + L^2/gamma_33) - beta^phi L.
//   T4  The interpolant exists where all four nodes do:  1 <= i <= n - 3 in both directions ("the domain").
//       An evaluation point (y0, an RK4 stage point, the end point of a step) outside the domain, or with a NaN
//       coordinate, ends the particle with status OUTSIDE = 4; that step is not taken.
//   T5  RK4, Kahan update (P1), stop rules B1-B6 and the equatorial-crossing event B5 exactly as in
//       geo_oracle.cpp with r -> x^1, theta -> x^2; per evaluation point the capture test comes first,
//       then the domain test.  Trajectory records (five-field path, round 2): S1-S3 of geo_oracle.cpp, components
//       (t, x1, x2, phi, E, p1, p2, L) selected by snap_mask; no Cartesian option (the coordinates are the table's own).
//
//   T6  (round 2) GENERAL stationary, axisymmetric 3+1 metric: all TEN functions of line element (1) --
//       alpha, beta^1, beta^2, beta^3, gamma_11, gamma_12, gamma_13, gamma_22, gamma_23, gamma_33 (x^3 = phi) -- of
//       (x^1, x^2), tab[f][j][i] in that order; no circularity, no diagonal 3-metric assumed (e.g. Kerr in horizon-
//       penetrating Kerr-Schild coordinates: beta^r != 0, gamma_r phi != 0).  Same interpolant (T2), domain (T4), stepper
//       and stop rules (T5).  With p = (p_1, p_2, L), gamma^{ij} the inverse of gamma_ij, V^i = gamma^{ij} p_j,
//       W = E + beta^k p_k, u^t = W / alpha^2:
//           H = 1/2 [ -W^2/alpha^2 + gamma^{ij} p_i p_j ]                                   (eq.(4) with eq.(1))
//           dt/dtau = u^t,   dx^i/dtau = V^i - beta^i u^t   (i = 1, 2, 3)
//           dp_k/dtau = -alpha (u^t)^2 d_k alpha + u^t p_j d_k beta^j + 1/2 V^a V^b d_k gamma_ab   (k = 1, 2);  dL/dtau = 0
//       (from d_k gamma^{ij} = -gamma^{ia} gamma^{jb} d_k gamma_ab), E = alpha sqrt(kappa + gamma^{ij} p_i p_j) - beta^k p_k.
//
// Pins (tests/test_oracle_tabulated.py): the interpolant against Keys' kernel form, node values, quadratic
// exactness, C^1 continuity; the RHS against finite differences of H on a metric with quadratic-polynomial
// fields (where the interpolant is exact); flat space in spherical coordinates against the straight line's
// closed form; tabulated Kerr against the pinned analytic-metric oracle with second-order convergence in
// the grid spacing; E, L exact and 2H drift.
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

enum { TAB_ST_MAXSTEPS = 0, TAB_ST_CAPTURED = 1, TAB_ST_ESCAPED = 2, TAB_ST_NUMERIC = 3, TAB_ST_OUTSIDE = 4 };
enum { F_ALPHA = 0, F_BETA = 1, F_G11 = 2, F_G22 = 3, F_G33 = 4 };

struct Table {
    const double* tab;   // [5][n2][n1]
    int64_t n1, n2;
    double x1_0, d1, x2_0, d2;
};

template <class R> struct Fields { R f[5], d1[5], d2[5]; };   // value, d/dx^1, d/dx^2 of the five fields

// T2: weights of nodes i-1, i, i+1, i+2 and their s-derivatives
template <class R> void keys_weights(R s, R w[4], R dw[4]) {
    const R s2 = s * s, s3 = s2 * s;
    w[0] = (-s3 + R(2) * s2 - s) / R(2);
    w[1] = (R(3) * s3 - R(5) * s2 + R(2)) / R(2);
    w[2] = (-R(3) * s3 + R(4) * s2 + s) / R(2);
    w[3] = (s3 - s2) / R(2);
    dw[0] = (-R(3) * s2 + R(4) * s - R(1)) / R(2);
    dw[1] = (R(9) * s2 - R(10) * s) / R(2);
    dw[2] = (-R(9) * s2 + R(8) * s + R(1)) / R(2);
    dw[3] = (R(3) * s2 - R(2) * s) / R(2);
}

// T2 + T4: false if (x1, x2) is outside the domain
template <class R> bool interpolate(const Table& m, R x1, R x2, Fields<R>& F) {
    const R u1 = (x1 - (R)m.x1_0) / (R)m.d1, u2 = (x2 - (R)m.x2_0) / (R)m.d2;
    const R fl1 = std::floor(u1), fl2 = std::floor(u2);
    if (!(fl1 >= R(1) && fl1 <= (R)(m.n1 - 3) && fl2 >= R(1) && fl2 <= (R)(m.n2 - 3))) return false;   // NaN-safe
    const int64_t i = (int64_t)fl1, j = (int64_t)fl2;
    R w1[4], dw1[4], w2[4], dw2[4];
    keys_weights(u1 - fl1, w1, dw1);
    keys_weights(u2 - fl2, w2, dw2);
    for (int f = 0; f < 5; ++f) {
        const double* T = m.tab + (int64_t)f * m.n1 * m.n2;
        R v = 0, v1 = 0, v2 = 0;
        for (int b = 0; b < 4; ++b)
            for (int a = 0; a < 4; ++a) {
                const R node = (R)T[(j - 1 + b) * m.n1 + (i - 1 + a)];
                v += w2[b] * w1[a] * node;
                v1 += w2[b] * dw1[a] * node;
                v2 += dw2[b] * w1[a] * node;
            }
        F.f[f] = v;
        F.d1[f] = v1 / (R)m.d1;
        F.d2[f] = v2 / (R)m.d2;
    }
    return true;
}

// State: y = (t, x1, x2, phi, E, p1, p2, L) -- the paper's order with r -> x^1, theta -> x^2
template <class R> struct State { R t, x1, x2, ph, E, p1, p2, L; };
template <class R> struct Deriv { R t, x1, x2, ph, p1, p2; };

// T3
template <class R> Deriv<R> rhs_fields(const Fields<R>& F, const State<R>& y) {
    const R al = F.f[F_ALPHA], be = F.f[F_BETA], g11 = F.f[F_G11], g22 = F.f[F_G22], g33 = F.f[F_G33];
    const R W = y.E + be * y.L;
    const R ut = W / (al * al);
    const R v1 = y.p1 / g11, v2 = y.p2 / g22, v3 = y.L / g33;
    Deriv<R> d;
    d.t = ut;
    d.x1 = v1;
    d.x2 = v2;
    d.ph = v3 - be * ut;
    d.p1 = ut * y.L * F.d1[F_BETA] - al * ut * ut * F.d1[F_ALPHA]
           + (F.d1[F_G11] * v1 * v1 + F.d1[F_G22] * v2 * v2 + F.d1[F_G33] * v3 * v3) / R(2);
    d.p2 = ut * y.L * F.d2[F_BETA] - al * ut * ut * F.d2[F_ALPHA]
           + (F.d2[F_G11] * v1 * v1 + F.d2[F_G22] * v2 * v2 + F.d2[F_G33] * v3 * v3) / R(2);
    return d;
}

template <class R> R hamiltonian_fields(const Fields<R>& F, const State<R>& y) {
    const R W = y.E + F.f[F_BETA] * y.L;
    return (-(W * W) / (F.f[F_ALPHA] * F.f[F_ALPHA]) + y.p1 * y.p1 / F.f[F_G11] + y.p2 * y.p2 / F.f[F_G22] +
            y.L * y.L / F.f[F_G33]) / R(2);
}

template <class R> R energy_fields(const Fields<R>& F, R p1, R p2, R L, R kappa) {
    return F.f[F_ALPHA] * std::sqrt(kappa + p1 * p1 / F.f[F_G11] + p2 * p2 / F.f[F_G22] + L * L / F.f[F_G33]) -
           F.f[F_BETA] * L;
}

struct StopRule { double r_capture, r_escape; int32_t kind; int32_t flags; };
struct OutPtrs {
    double* final_state; int32_t* status; int64_t* steps_done; double* eq_cross_r; double* health;
    // trajectory records (five-field path only, round 2): as in geo_oracle.cpp, readings S1-S3
    double* snapshots;      // [n][snap_capacity][ncomp] or null
    int64_t snap_capacity;
    uint32_t snap_mask;     // bit k: component k of (t, x1, x2, phi, E, p1, p2, L)
    int32_t* snap_count;    // [n] or null
};

template <class R> struct State;
template <class R>
void write_record(const OutPtrs& o, int64_t i, int64_t slot, const R comp[8]) {
    if (!o.snapshots || slot >= o.snap_capacity) return;   // S3: drop, never overflow
    int ncomp = 0;
    for (int k = 0; k < 8; ++k) ncomp += (o.snap_mask >> k) & 1u;
    double* dst = o.snapshots + (i * o.snap_capacity + slot) * ncomp;
    int j = 0;
    for (int k = 0; k < 8; ++k)
        if ((o.snap_mask >> k) & 1u) dst[j++] = (double)comp[k];
}

template <class R> bool finite6(const State<R>& y) {
    return std::isfinite(y.t) && std::isfinite(y.x1) && std::isfinite(y.x2) && std::isfinite(y.ph) &&
           std::isfinite(y.p1) && std::isfinite(y.p2);
}

template <class R> State<R> shifted(const State<R>& y, R w, const Deriv<R>& k) {
    State<R> z = y;
    z.t = y.t + w * k.t;
    z.x1 = y.x1 + w * k.x1;
    z.x2 = y.x2 + w * k.x2;
    z.ph = y.ph + w * k.ph;
    z.p1 = y.p1 + w * k.p1;
    z.p2 = y.p2 + w * k.p2;
    return z;
}

template <class R> void kahan_add(R& y, R& c, R delta, bool plain) {
    if (plain) { y = y + delta; return; }
    const R yk = delta - c;
    const R tsum = y + yk;
    c = (tsum - y) - yk;
    y = tsum;
}

template <class R>
void integrate_one(const Table& m, const double* state_in, int64_t n, int64_t i, R h, int64_t nsteps,
                   const StopRule& st, const OutPtrs& o, int64_t snapshot_every = 0) {
    const R kappa = st.kind == 0 ? R(1) : R(0);
    const bool plain = (st.flags & 1) != 0;
    const R rc = (R)st.r_capture, re = (R)st.r_escape;
    const R half_pi = (R)1.5707963267948966;

    State<R> y;
    y.t = R(0);
    y.x1 = (R)state_in[0 * n + i];
    y.x2 = (R)state_in[1 * n + i];
    y.ph = (R)state_in[2 * n + i];
    y.p1 = (R)state_in[3 * n + i];
    y.p2 = (R)state_in[4 * n + i];
    y.L = (R)state_in[5 * n + i];
    y.E = std::numeric_limits<R>::quiet_NaN();
    R ct = 0, c1 = 0, c2 = 0, cph = 0, cp1 = 0, cp2 = 0;

    int32_t status = -1;
    int64_t steps = 0, snaps = 0;
    R eq_cross = std::numeric_limits<R>::quiet_NaN();
    bool crossed = false;
    Fields<R> F;
    auto record = [&]() {
        const R comp[8] = {y.t, y.x1, y.x2, y.ph, y.E, y.p1, y.p2, y.L};
        write_record<R>(o, i, snaps, comp);
        ++snaps;
    };

    // B1 + T4 on y0
    if (!(y.x1 >= rc)) status = TAB_ST_CAPTURED;
    else if (!finite6(y) || !std::isfinite(y.L)) status = TAB_ST_NUMERIC;
    else if (!interpolate(m, y.x1, y.x2, F)) status = TAB_ST_OUTSIDE;
    else {
        y.E = energy_fields(F, y.p1, y.p2, y.L, kappa);
        if (!std::isfinite(y.E)) status = TAB_ST_NUMERIC;
        else {
            if (snapshot_every > 0) record();                        // S1: slot 0 = y0 (E known: it passed every y0 test)
            if (y.x1 > re) status = TAB_ST_ESCAPED;
            else if (nsteps == 0) status = TAB_ST_MAXSTEPS;
        }
    }

    while (status < 0) {
        // F holds the fields at y (from B1 or from the end point test of the previous step)
        const Deriv<R> k1 = rhs_fields(F, y);
        const State<R> y2 = shifted(y, h / R(2), k1);
        Fields<R> G;
        if (!(y2.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!interpolate(m, y2.x1, y2.x2, G)) { status = TAB_ST_OUTSIDE; break; }
        const Deriv<R> k2 = rhs_fields(G, y2);
        const State<R> y3 = shifted(y, h / R(2), k2);
        if (!(y3.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!interpolate(m, y3.x1, y3.x2, G)) { status = TAB_ST_OUTSIDE; break; }
        const Deriv<R> k3 = rhs_fields(G, y3);
        const State<R> y4 = shifted(y, h, k3);
        if (!(y4.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!interpolate(m, y4.x1, y4.x2, G)) { status = TAB_ST_OUTSIDE; break; }
        const Deriv<R> k4 = rhs_fields(G, y4);

        State<R> yn = y;
        R nt = ct, n1 = c1, n2 = c2, nph = cph, np1 = cp1, np2 = cp2;
        const R w = h / R(6);
        kahan_add(yn.t, nt, w * (k1.t + R(2) * k2.t + R(2) * k3.t + k4.t), plain);
        kahan_add(yn.x1, n1, w * (k1.x1 + R(2) * k2.x1 + R(2) * k3.x1 + k4.x1), plain);
        kahan_add(yn.x2, n2, w * (k1.x2 + R(2) * k2.x2 + R(2) * k3.x2 + k4.x2), plain);
        kahan_add(yn.ph, nph, w * (k1.ph + R(2) * k2.ph + R(2) * k3.ph + k4.ph), plain);
        kahan_add(yn.p1, np1, w * (k1.p1 + R(2) * k2.p1 + R(2) * k3.p1 + k4.p1), plain);
        kahan_add(yn.p2, np2, w * (k1.p2 + R(2) * k2.p2 + R(2) * k3.p2 + k4.p2), plain);

        if (!(yn.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!finite6(yn)) { status = TAB_ST_NUMERIC; break; }
        if (!interpolate(m, yn.x1, yn.x2, G)) { status = TAB_ST_OUTSIDE; break; }     // T4: end point

        if (!crossed) {
            const R d0 = y.x2 - half_pi, d1 = yn.x2 - half_pi;
            if (d0 * d1 < R(0)) {
                crossed = true;
                eq_cross = y.x1 + (yn.x1 - y.x1) * (half_pi - y.x2) / (yn.x2 - y.x2);
            }
        }
        y = yn; ct = nt; c1 = n1; c2 = n2; cph = nph; cp1 = np1; cp2 = np2;
        F = G;
        ++steps;
        if (snapshot_every > 0 && steps % snapshot_every == 0) record();   // S1
        if (y.x1 > re) status = TAB_ST_ESCAPED;
        else if (steps >= nsteps) status = TAB_ST_MAXSTEPS;
    }

    const R comp[8] = {y.t, y.x1, y.x2, y.ph, y.E, y.p1, y.p2, y.L};
    for (int k = 0; k < 8; ++k) o.final_state[(int64_t)k * n + i] = (double)comp[k];
    o.status[i] = status;
    o.steps_done[i] = steps;
    if (o.eq_cross_r) o.eq_cross_r[i] = (double)eq_cross;
    if (snapshot_every > 0 && o.snap_count) o.snap_count[i] = (int32_t)snaps;
    if (o.health) {
        // |2H + kappa| of the final state; NaN where the final state has no interpolant (OUTSIDE at y0, NUMERIC)
        Fields<R> H;
        o.health[i] = (std::isfinite(y.E) && interpolate(m, y.x1, y.x2, H))
                          ? (double)std::fabs(R(2) * hamiltonian_fields(H, y) + kappa)
                          : std::numeric_limits<double>::quiet_NaN();
    }
}

template <class R>
void integrate_range(const Table& m, const double* state_in, int64_t n, double h, int64_t nsteps,
                     const StopRule& st, const OutPtrs& o, int64_t lo, int64_t hi, int64_t snapshot_every) {
    for (int64_t i = lo; i < hi; ++i) integrate_one<R>(m, state_in, n, i, (R)h, nsteps, st, o, snapshot_every);
}


// ---------------------------------------------------------------------------------------------------------------
// T7 (round 2): the adaptive Dormand-Prince 5(4) stepper of readings A1-A3 on a tabulated metric -- five fields (MP = Metric5:
// the T3 right-hand side) or all ten (MP = Metric10: the T6 right-hand side); the policy only names which interpolate / rhs /
// energy / hamiltonian routines of this file are called.
// The loop of geo_oracle.cpp: integrate_one_adaptive with r -> x^1, theta -> x^2 and the T3 right-hand side; in addition
// every evaluation point (y0, the six stage points, the end point) is tested against the table's domain (T4): per point
// the capture test comes first, then the domain test; the first event in evaluation order ends the particle
// (CAPTURED / OUTSIDE), that attempt is not taken.
// ---------------------------------------------------------------------------------------------------------------
template <class R> R tcomp6(const State<R>& y, int c) {
    switch (c) { case 0: return y.t; case 1: return y.x1; case 2: return y.x2; case 3: return y.ph; case 4: return y.p1; default: return y.p2; }
}
template <class R> R tdcomp6(const Deriv<R>& k, int c) {
    switch (c) { case 0: return k.t; case 1: return k.x1; case 2: return k.x2; case 3: return k.ph; case 4: return k.p1; default: return k.p2; }
}
template <class R> void tset6(State<R>& y, int c, R v) {
    switch (c) { case 0: y.t = v; break; case 1: y.x1 = v; break; case 2: y.x2 = v; break; case 3: y.ph = v; break;
                 case 4: y.p1 = v; break; default: y.p2 = v; }
}

template <class R, class MP>
void integrate_one_adaptive_tab(const Table& m, const double* state_in, int64_t n, int64_t i, const AdaptiveCtl& ctl,
                                int64_t max_attempts, const StopRule& st, const OutPtrs& o, int64_t* rejected_out) {
    static const DP45 T;
    const R kappa = st.kind == 0 ? R(1) : R(0);
    const R rc = (R)st.r_capture, re = (R)st.r_escape;
    const R half_pi = (R)1.5707963267948966;
    State<R> y;
    y.t = R(0);
    y.x1 = (R)state_in[0 * n + i];
    y.x2 = (R)state_in[1 * n + i];
    y.ph = (R)state_in[2 * n + i];
    y.p1 = (R)state_in[3 * n + i];
    y.p2 = (R)state_in[4 * n + i];
    y.L = (R)state_in[5 * n + i];
    y.E = std::numeric_limits<R>::quiet_NaN();
    R cc[6] = {0, 0, 0, 0, 0, 0};
    R h = (R)ctl.h0, tau = R(0);
    const R tau_end = (R)ctl.tau_end;
    const bool dense = ctl.snap_dtau > 0.0 && o.snapshots != nullptr;
    const R dtau = (R)ctl.snap_dtau;
    int64_t next_j = 0;
    int32_t status = -1;
    int64_t steps = 0, attempts = 0, rejected = 0;
    R eq_cross = std::numeric_limits<R>::quiet_NaN();
    bool crossed = false;
    typename MP::F F;
    auto record = [&](const State<R>& ys) {
        const R comp[8] = {ys.t, ys.x1, ys.x2, ys.ph, ys.E, ys.p1, ys.p2, ys.L};
        write_record<R>(o, i, next_j, comp);
        ++next_j;
    };
    if (!(y.x1 >= rc)) status = TAB_ST_CAPTURED;                     // B1 + T4 on y0
    else if (!finite6(y) || !std::isfinite(y.L)) status = TAB_ST_NUMERIC;
    else if (!MP::interp(m, y.x1, y.x2, F)) status = TAB_ST_OUTSIDE;
    else {
        y.E = MP::energy(F, y.p1, y.p2, y.L, kappa);
        if (!std::isfinite(y.E)) status = TAB_ST_NUMERIC;
        else {
            if (dense) record(y);
            if (y.x1 > re) status = TAB_ST_ESCAPED;
            else if (max_attempts == 0) status = TAB_ST_MAXSTEPS;
        }
    }
    Deriv<R> k[DP45::S];
    if (status < 0) k[0] = MP::rhs(F, y);
    while (status < 0) {
        const bool last = tau + R(1.01) * h >= tau_end;
        if (last) h = tau_end - tau;
        int ev = 0;
        for (int s = 1; s < DP45::S - 1 && !ev; ++s) {               // stages 2..6
            State<R> ys = y;
            for (int c = 0; c < 6; ++c) {
                R acc = R(0);
                for (int j = 0; j < s; ++j) acc += (R)T.a[s][j] * tdcomp6(k[j], c);
                tset6(ys, c, tcomp6(y, c) + h * acc);
            }
            typename MP::F G;
            if (!(ys.x1 >= rc)) ev = TAB_ST_CAPTURED;
            else if (!MP::interp(m, ys.x1, ys.x2, G)) ev = TAB_ST_OUTSIDE;
            else k[s] = MP::rhs(G, ys);
        }
        ++attempts;
        if (ev) { status = ev; break; }
        State<R> yn = y;
        R cn[6];
        for (int c = 0; c < 6; ++c) {
            R acc5 = R(0);
            for (int j = 0; j < DP45::S - 1; ++j) acc5 += (R)T.a[6][j] * tdcomp6(k[j], c);
            R v = tcomp6(y, c);
            cn[c] = cc[c];
            kahan_add(v, cn[c], h * acc5, false);
            tset6(yn, c, v);
        }
        if (!(yn.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }     // end point: capture, then finiteness, then domain
        const bool fin = finite6(yn);
        typename MP::F Gn;
        if (fin && !MP::interp(m, yn.x1, yn.x2, Gn)) { status = TAB_ST_OUTSIDE; break; }
        R err = R(0);
        if (fin) {
            k[6] = MP::rhs(Gn, yn);
            for (int c = 0; c < 6; ++c) {
                R acce = R(0);
                for (int j = 0; j < DP45::S; ++j)
                    acce += ((R)(j < 6 ? T.a[6][j] : 0.0L) - (R)T.b4[j]) * tdcomp6(k[j], c);
                const R sc = (R)ctl.atol + (R)ctl.rtol * std::max(std::fabs(tcomp6(y, c)), std::fabs(tcomp6(yn, c)));
                const R ec = std::fabs(h * acce) / sc;
                if (!(ec <= err)) err = ec;
            }
        }
        if (fin && std::isinf(ctl.rtol)) err = R(0);
        R fac = err > R(0) ? R(0.9) * std::pow(err, R(-0.2)) : (err == R(0) ? R(5) : R(0.2));
        if (!(fac >= R(0.2))) fac = R(0.2);
        if (fac > R(5)) fac = R(5);
        if (std::isinf(ctl.rtol)) fac = R(1);
        if (!fin || !(err <= R(1))) {
            ++rejected;
            h *= std::min(fac, R(1));
            if ((std::isinf(ctl.rtol) && !fin) || !(std::fabs(h) >= (R)ctl.h_min) || !(std::fabs(h) > R(0))) { status = TAB_ST_NUMERIC; break; }
            if (attempts >= max_attempts) { status = TAB_ST_MAXSTEPS; break; }
            continue;
        }
        if (!crossed) {
            const R d0 = y.x2 - half_pi, d1 = yn.x2 - half_pi;
            if (d0 * d1 < R(0)) {
                crossed = true;
                eq_cross = y.x1 + (yn.x1 - y.x1) * (half_pi - y.x2) / (yn.x2 - y.x2);
            }
        }
        const R tau_new = last ? tau_end : tau + h;
        if (dense) {
            for (;;) {
                const R tj = (R)next_j * dtau;
                if (!(tj <= tau_new)) break;
                R w[7];
                dp45_dense_weights<R>((tj - tau) / h, w);
                State<R> ys = y;
                for (int c = 0; c < 6; ++c) {
                    R acc = R(0);
                    for (int j = 0; j < DP45::S; ++j) acc += w[j] * tdcomp6(k[j], c);
                    tset6(ys, c, tcomp6(y, c) + h * acc);
                }
                record(ys);
            }
        }
        y = yn;
        for (int c = 0; c < 6; ++c) cc[c] = cn[c];
        k[0] = k[6];
        F = Gn;
        ++steps;
        tau = tau_new;
        h *= fac;
        if (y.x1 > re) status = TAB_ST_ESCAPED;
        else if (last || attempts >= max_attempts) status = TAB_ST_MAXSTEPS;
    }
    const R comp[8] = {y.t, y.x1, y.x2, y.ph, y.E, y.p1, y.p2, y.L};
    for (int q = 0; q < 8; ++q) o.final_state[(int64_t)q * n + i] = (double)comp[q];
    o.status[i] = status;
    o.steps_done[i] = steps;
    if (o.eq_cross_r) o.eq_cross_r[i] = (double)eq_cross;
    if (o.health) {
        typename MP::F H;
        o.health[i] = (std::isfinite(y.E) && MP::interp(m, y.x1, y.x2, H))
                          ? (double)std::fabs(R(2) * MP::hamiltonian(H, y) + kappa)
                          : std::numeric_limits<double>::quiet_NaN();
    }
    if (dense && o.snap_count) o.snap_count[i] = (int32_t)next_j;
    if (rejected_out) rejected_out[i] = rejected;
}

// ---------------------------------------------------------------------------------------------------------------
// T6: general stationary axisymmetric 3+1 metric, ten fields
// ---------------------------------------------------------------------------------------------------------------
enum { G_ALPHA = 0, G_B1 = 1, G_B2 = 2, G_B3 = 3, G_G11 = 4, G_G12 = 5, G_G13 = 6, G_G22 = 7, G_G23 = 8, G_G33 = 9, G_NF = 10 };
template <class R> struct GFields { R f[G_NF], d1[G_NF], d2[G_NF]; };

template <class R> bool interpolate_general(const Table& m, R x1, R x2, GFields<R>& F) {
    const R u1 = (x1 - (R)m.x1_0) / (R)m.d1, u2 = (x2 - (R)m.x2_0) / (R)m.d2;
    const R fl1 = std::floor(u1), fl2 = std::floor(u2);
    if (!(fl1 >= R(1) && fl1 <= (R)(m.n1 - 3) && fl2 >= R(1) && fl2 <= (R)(m.n2 - 3))) return false;
    const int64_t i = (int64_t)fl1, j = (int64_t)fl2;
    R w1[4], dw1[4], w2[4], dw2[4];
    keys_weights(u1 - fl1, w1, dw1);
    keys_weights(u2 - fl2, w2, dw2);
    for (int f = 0; f < G_NF; ++f) {
        const double* T = m.tab + (int64_t)f * m.n1 * m.n2;
        R v = 0, v1 = 0, v2 = 0;
        for (int b = 0; b < 4; ++b)
            for (int a = 0; a < 4; ++a) {
                const R node = (R)T[(j - 1 + b) * m.n1 + (i - 1 + a)];
                v += w2[b] * w1[a] * node;
                v1 += w2[b] * dw1[a] * node;
                v2 += dw2[b] * w1[a] * node;
            }
        F.f[f] = v;
        F.d1[f] = v1 / (R)m.d1;
        F.d2[f] = v2 / (R)m.d2;
    }
    return true;
}

// gamma^{ij} (symmetric 3 x 3 inverse by the adjugate) as [11, 12, 13, 22, 23, 33]
template <class R> void inverse3(const R* f, R gi[6]) {
    const R a = f[G_G11], b = f[G_G12], c = f[G_G13], d = f[G_G22], e = f[G_G23], g = f[G_G33];
    const R c11 = d * g - e * e, c12 = c * e - b * g, c13 = b * e - c * d;
    const R det = a * c11 + b * c12 + c * c13;
    gi[0] = c11 / det; gi[1] = c12 / det; gi[2] = c13 / det;
    gi[3] = (a * g - c * c) / det; gi[4] = (b * c - a * e) / det; gi[5] = (a * d - b * b) / det;
}

template <class R> struct GAux { R V[3], W, ut, gpp; };     // V^i, W, u^t, gamma^{ij} p_i p_j
template <class R> GAux<R> aux_general(const GFields<R>& F, R p1, R p2, R L, R E) {
    R gi[6];
    inverse3(F.f, gi);
    GAux<R> A;
    A.V[0] = gi[0] * p1 + gi[1] * p2 + gi[2] * L;
    A.V[1] = gi[1] * p1 + gi[3] * p2 + gi[4] * L;
    A.V[2] = gi[2] * p1 + gi[4] * p2 + gi[5] * L;
    A.gpp = A.V[0] * p1 + A.V[1] * p2 + A.V[2] * L;
    A.W = E + F.f[G_B1] * p1 + F.f[G_B2] * p2 + F.f[G_B3] * L;
    A.ut = A.W / (F.f[G_ALPHA] * F.f[G_ALPHA]);
    return A;
}

template <class R> Deriv<R> rhs_general(const GFields<R>& F, const State<R>& y) {
    const GAux<R> A = aux_general(F, y.p1, y.p2, y.L, y.E);
    const R al = F.f[G_ALPHA];
    Deriv<R> d;
    d.t = A.ut;
    d.x1 = A.V[0] - F.f[G_B1] * A.ut;
    d.x2 = A.V[1] - F.f[G_B2] * A.ut;
    d.ph = A.V[2] - F.f[G_B3] * A.ut;
    const R* D[2] = {F.d1, F.d2};
    R dp[2];
    for (int k = 0; k < 2; ++k) {
        const R* q = D[k];
        const R VVdg = A.V[0] * A.V[0] * q[G_G11] + A.V[1] * A.V[1] * q[G_G22] + A.V[2] * A.V[2] * q[G_G33] +
                       R(2) * (A.V[0] * A.V[1] * q[G_G12] + A.V[0] * A.V[2] * q[G_G13] + A.V[1] * A.V[2] * q[G_G23]);
        dp[k] = -al * A.ut * A.ut * q[G_ALPHA] + A.ut * (y.p1 * q[G_B1] + y.p2 * q[G_B2] + y.L * q[G_B3]) + VVdg / R(2);
    }
    d.p1 = dp[0];
    d.p2 = dp[1];
    return d;
}

template <class R> R hamiltonian_general(const GFields<R>& F, const State<R>& y) {
    const GAux<R> A = aux_general(F, y.p1, y.p2, y.L, y.E);
    return (-(A.W * A.W) / (F.f[G_ALPHA] * F.f[G_ALPHA]) + A.gpp) / R(2);
}

template <class R> R energy_general(const GFields<R>& F, R p1, R p2, R L, R kappa) {
    const GAux<R> A = aux_general(F, p1, p2, L, R(0));
    return F.f[G_ALPHA] * std::sqrt(kappa + A.gpp) - (F.f[G_B1] * p1 + F.f[G_B2] * p2 + F.f[G_B3] * L);
}

// T5 with the T6 right-hand side: the loop of integrate_one, written out again for the general fields
template <class R>
void integrate_one_general(const Table& m, const double* state_in, int64_t n, int64_t i, R h, int64_t nsteps,
                           const StopRule& st, const OutPtrs& o, int64_t snapshot_every = 0) {
    const R kappa = st.kind == 0 ? R(1) : R(0);
    const bool plain = (st.flags & 1) != 0;
    const R rc = (R)st.r_capture, re = (R)st.r_escape;
    const R half_pi = (R)1.5707963267948966;
    State<R> y;
    y.t = R(0);
    y.x1 = (R)state_in[0 * n + i];
    y.x2 = (R)state_in[1 * n + i];
    y.ph = (R)state_in[2 * n + i];
    y.p1 = (R)state_in[3 * n + i];
    y.p2 = (R)state_in[4 * n + i];
    y.L = (R)state_in[5 * n + i];
    y.E = std::numeric_limits<R>::quiet_NaN();
    R ct = 0, c1 = 0, c2 = 0, cph = 0, cp1 = 0, cp2 = 0;
    int32_t status = -1;
    int64_t steps = 0, snaps = 0;
    R eq_cross = std::numeric_limits<R>::quiet_NaN();
    bool crossed = false;
    GFields<R> F;
    auto record = [&]() {                                            // S1-S3, as on the five-field path
        const R comp[8] = {y.t, y.x1, y.x2, y.ph, y.E, y.p1, y.p2, y.L};
        write_record<R>(o, i, snaps, comp);
        ++snaps;
    };
    if (!(y.x1 >= rc)) status = TAB_ST_CAPTURED;
    else if (!finite6(y) || !std::isfinite(y.L)) status = TAB_ST_NUMERIC;
    else if (!interpolate_general(m, y.x1, y.x2, F)) status = TAB_ST_OUTSIDE;
    else {
        y.E = energy_general(F, y.p1, y.p2, y.L, kappa);
        if (!std::isfinite(y.E)) status = TAB_ST_NUMERIC;
        else {
            if (snapshot_every > 0) record();
            if (y.x1 > re) status = TAB_ST_ESCAPED;
            else if (nsteps == 0) status = TAB_ST_MAXSTEPS;
        }
    }
    while (status < 0) {
        const Deriv<R> k1 = rhs_general(F, y);
        const State<R> y2 = shifted(y, h / R(2), k1);
        GFields<R> G;
        if (!(y2.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!interpolate_general(m, y2.x1, y2.x2, G)) { status = TAB_ST_OUTSIDE; break; }
        const Deriv<R> k2 = rhs_general(G, y2);
        const State<R> y3 = shifted(y, h / R(2), k2);
        if (!(y3.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!interpolate_general(m, y3.x1, y3.x2, G)) { status = TAB_ST_OUTSIDE; break; }
        const Deriv<R> k3 = rhs_general(G, y3);
        const State<R> y4 = shifted(y, h, k3);
        if (!(y4.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!interpolate_general(m, y4.x1, y4.x2, G)) { status = TAB_ST_OUTSIDE; break; }
        const Deriv<R> k4 = rhs_general(G, y4);
        State<R> yn = y;
        R nt = ct, n1 = c1, n2 = c2, nph = cph, np1 = cp1, np2 = cp2;
        const R w = h / R(6);
        kahan_add(yn.t, nt, w * (k1.t + R(2) * k2.t + R(2) * k3.t + k4.t), plain);
        kahan_add(yn.x1, n1, w * (k1.x1 + R(2) * k2.x1 + R(2) * k3.x1 + k4.x1), plain);
        kahan_add(yn.x2, n2, w * (k1.x2 + R(2) * k2.x2 + R(2) * k3.x2 + k4.x2), plain);
        kahan_add(yn.ph, nph, w * (k1.ph + R(2) * k2.ph + R(2) * k3.ph + k4.ph), plain);
        kahan_add(yn.p1, np1, w * (k1.p1 + R(2) * k2.p1 + R(2) * k3.p1 + k4.p1), plain);
        kahan_add(yn.p2, np2, w * (k1.p2 + R(2) * k2.p2 + R(2) * k3.p2 + k4.p2), plain);
        if (!(yn.x1 >= rc)) { status = TAB_ST_CAPTURED; break; }
        if (!finite6(yn)) { status = TAB_ST_NUMERIC; break; }
        if (!interpolate_general(m, yn.x1, yn.x2, G)) { status = TAB_ST_OUTSIDE; break; }
        if (!crossed) {
            const R d0 = y.x2 - half_pi, d1 = yn.x2 - half_pi;
            if (d0 * d1 < R(0)) {
                crossed = true;
                eq_cross = y.x1 + (yn.x1 - y.x1) * (half_pi - y.x2) / (yn.x2 - y.x2);
            }
        }
        y = yn; ct = nt; c1 = n1; c2 = n2; cph = nph; cp1 = np1; cp2 = np2;
        F = G;
        ++steps;
        if (snapshot_every > 0 && steps % snapshot_every == 0) record();
        if (y.x1 > re) status = TAB_ST_ESCAPED;
        else if (steps >= nsteps) status = TAB_ST_MAXSTEPS;
    }
    const R comp[8] = {y.t, y.x1, y.x2, y.ph, y.E, y.p1, y.p2, y.L};
    for (int k = 0; k < 8; ++k) o.final_state[(int64_t)k * n + i] = (double)comp[k];
    o.status[i] = status;
    o.steps_done[i] = steps;
    if (o.eq_cross_r) o.eq_cross_r[i] = (double)eq_cross;
    if (snapshot_every > 0 && o.snap_count) o.snap_count[i] = (int32_t)snaps;
    if (o.health) {
        GFields<R> H;
        o.health[i] = (std::isfinite(y.E) && interpolate_general(m, y.x1, y.x2, H))
                          ? (double)std::fabs(R(2) * hamiltonian_general(H, y) + kappa)
                          : std::numeric_limits<double>::quiet_NaN();
    }
}

template <class R>
void integrate_range_general(const Table& m, const double* state_in, int64_t n, double h, int64_t nsteps,
                             const StopRule& st, const OutPtrs& o, int64_t lo, int64_t hi, int64_t snapshot_every) {
    for (int64_t i = lo; i < hi; ++i) integrate_one_general<R>(m, state_in, n, i, (R)h, nsteps, st, o, snapshot_every);
}

// the two metric policies of integrate_one_adaptive_tab
template <class R> struct Metric5 {
    typedef Fields<R> F;
    static bool interp(const Table& m, R x1, R x2, F& f) { return interpolate(m, x1, x2, f); }
    static Deriv<R> rhs(const F& f, const State<R>& y) { return rhs_fields(f, y); }
    static R energy(const F& f, R p1, R p2, R L, R kappa) { return energy_fields(f, p1, p2, L, kappa); }
    static R hamiltonian(const F& f, const State<R>& y) { return hamiltonian_fields(f, y); }
};
template <class R> struct Metric10 {
    typedef GFields<R> F;
    static bool interp(const Table& m, R x1, R x2, F& f) { return interpolate_general(m, x1, x2, f); }
    static Deriv<R> rhs(const F& f, const State<R>& y) { return rhs_general(f, y); }
    static R energy(const F& f, R p1, R p2, R L, R kappa) { return energy_general(f, p1, p2, L, kappa); }
    static R hamiltonian(const F& f, const State<R>& y) { return hamiltonian_general(f, y); }
};

}  // namespace

extern "C" {

// tab: [5][n2][n1] host doubles.  precision: 0 = double, 1 = long double.  Returns 0, or 1 on invalid arguments.
int oracle_tab_integrate(const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                         const double* state_in, int64_t n, double h, int64_t nsteps, const StopRule* st,
                         const OutPtrs* out, int precision, int nthreads, int64_t snapshot_every) {
    if (!tab || n1 < 4 || n2 < 4 || !(d1 > 0) || !(d2 > 0) || n < 0 || nsteps < 0 || !st || !out || snapshot_every < 0) return 1;
    if (snapshot_every > 0 && (!out->snapshots || !out->snap_count || out->snap_capacity < 1 || (out->snap_mask & 0xFFu) == 0)) return 1;
    const Table m{tab, n1, n2, x1_0, d1, x2_0, d2};
    if (nthreads < 1) nthreads = 1;
    std::vector<std::thread> pool;
    const int64_t per = (n + nthreads - 1) / nthreads;
    for (int t = 0; t < nthreads; ++t) {
        const int64_t lo = t * per, hi = std::min<int64_t>(n, lo + per);
        if (lo >= hi) break;
        if (precision == 1)
            pool.emplace_back(integrate_range<long double>, m, state_in, n, h, nsteps, *st, *out, lo, hi, snapshot_every);
        else
            pool.emplace_back(integrate_range<double>, m, state_in, n, h, nsteps, *st, *out, lo, hi, snapshot_every);
    }
    for (auto& th : pool) th.join();
    return 0;
}

// Interpolated fields at one point: out15 = value[5], d/dx1[5], d/dx2[5].  Returns 1 inside the domain, 0 outside.
int oracle_tab_fields(const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                      double x1, double x2, double* out15) {
    const Table m{tab, n1, n2, x1_0, d1, x2_0, d2};
    Fields<double> F;
    if (!interpolate<double>(m, x1, x2, F)) return 0;
    for (int f = 0; f < 5; ++f) { out15[f] = F.f[f]; out15[5 + f] = F.d1[f]; out15[10 + f] = F.d2[f]; }
    return 1;
}

// RHS (T3) at y8 = (t, x1, x2, phi, E, p1, p2, L): d6 = d/dtau of (t, x1, x2, phi, p1, p2); *H = Hamiltonian.
int oracle_tab_rhs(const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                   const double* y8, double* d6, double* H) {
    const Table m{tab, n1, n2, x1_0, d1, x2_0, d2};
    Fields<double> F;
    State<double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
    if (!interpolate<double>(m, y.x1, y.x2, F)) return 0;
    const Deriv<double> d = rhs_fields(F, y);
    d6[0] = d.t; d6[1] = d.x1; d6[2] = d.x2; d6[3] = d.ph; d6[4] = d.p1; d6[5] = d.p2;
    if (H) *H = hamiltonian_fields(F, y);
    return 1;
}

// ---- T6: general ten-field tables, tab = [10][n2][n1] ----
int oracle_tabg_integrate(const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                          const double* state_in, int64_t n, double h, int64_t nsteps, const StopRule* st,
                          const OutPtrs* out, int precision, int nthreads, int64_t snapshot_every) {
    if (!tab || n1 < 4 || n2 < 4 || !(d1 > 0) || !(d2 > 0) || n < 0 || nsteps < 0 || !st || !out || snapshot_every < 0) return 1;
    if (snapshot_every > 0 && (!out->snapshots || !out->snap_count || out->snap_capacity < 1 || (out->snap_mask & 0xFFu) == 0)) return 1;
    const Table m{tab, n1, n2, x1_0, d1, x2_0, d2};
    if (nthreads < 1) nthreads = 1;
    std::vector<std::thread> pool;
    const int64_t per = (n + nthreads - 1) / nthreads;
    for (int t = 0; t < nthreads; ++t) {
        const int64_t lo = t * per, hi = std::min<int64_t>(n, lo + per);
        if (lo >= hi) break;
        if (precision == 1)
            pool.emplace_back(integrate_range_general<long double>, m, state_in, n, h, nsteps, *st, *out, lo, hi, snapshot_every);
        else
            pool.emplace_back(integrate_range_general<double>, m, state_in, n, h, nsteps, *st, *out, lo, hi, snapshot_every);
    }
    for (auto& th : pool) th.join();
    return 0;
}

// RHS (T6) at y8 = (t, x1, x2, phi, E, p1, p2, L): d6 = d/dtau of (t, x1, x2, phi, p1, p2); *H = Hamiltonian;
// E_out (optional) = mass-shell energy for kappa.  Returns 1 inside the domain, 0 outside.
int oracle_tabg_rhs(const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                    const double* y8, double* d6, double* H, double kappa, double* E_out) {
    const Table m{tab, n1, n2, x1_0, d1, x2_0, d2};
    GFields<double> F;
    State<double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
    if (!interpolate_general<double>(m, y.x1, y.x2, F)) return 0;
    const Deriv<double> d = rhs_general(F, y);
    d6[0] = d.t; d6[1] = d.x1; d6[2] = d.x2; d6[3] = d.ph; d6[4] = d.p1; d6[5] = d.p2;
    if (H) *H = hamiltonian_general(F, y);
    if (E_out) *E_out = energy_general(F, y.p1, y.p2, y.L, kappa);
    return 1;
}

// ---- T7: adaptive RK5(4) on a five-field table (general = 0) or a ten-field table (general = 1) ----
static int tab_integrate_adaptive(int general, const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                                  const double* state_in, int64_t n, const AdaptiveCtl* ctl, int64_t max_attempts,
                                  const StopRule* st, const OutPtrs* out, int64_t* rejected, int precision, int nthreads) {
    if (!tab || n1 < 4 || n2 < 4 || !(d1 > 0) || !(d2 > 0) || n < 0 || max_attempts < 0 || !st || !out || !ctl) return 1;
    if (!std::isfinite(ctl->h0) || !(ctl->h0 > 0.0) || !(ctl->rtol >= 0) || !(ctl->atol >= 0) || !(ctl->rtol + ctl->atol > 0) ||
        !(ctl->h_min >= 0) || !(ctl->tau_end > 0) || !(ctl->snap_dtau >= 0)) return 1;
    if (ctl->snap_dtau > 0 && (!out->snapshots || !out->snap_count || out->snap_capacity < 1 || (out->snap_mask & 0xFFu) == 0)) return 1;
    const Table m{tab, n1, n2, x1_0, d1, x2_0, d2};
    if (nthreads < 1) nthreads = 1;
    std::vector<std::thread> pool;
    const int64_t block = 64, nblocks = (n + block - 1) / block;
    for (int t = 0; t < nthreads; ++t)
        pool.emplace_back([&, t]() {
            for (int64_t b = t; b < nblocks; b += nthreads)
                for (int64_t i = b * block; i < std::min<int64_t>(n, (b + 1) * block); ++i) {
                    if (general) {
                        if (precision == 1) integrate_one_adaptive_tab<long double, Metric10<long double>>(m, state_in, n, i, *ctl, max_attempts, *st, *out, rejected);
                        else integrate_one_adaptive_tab<double, Metric10<double>>(m, state_in, n, i, *ctl, max_attempts, *st, *out, rejected);
                    } else {
                        if (precision == 1) integrate_one_adaptive_tab<long double, Metric5<long double>>(m, state_in, n, i, *ctl, max_attempts, *st, *out, rejected);
                        else integrate_one_adaptive_tab<double, Metric5<double>>(m, state_in, n, i, *ctl, max_attempts, *st, *out, rejected);
                    }
                }
        });
    for (auto& th : pool) th.join();
    return 0;
}

int oracle_tab_integrate_adaptive(const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                                  const double* state_in, int64_t n, const AdaptiveCtl* ctl, int64_t max_attempts,
                                  const StopRule* st, const OutPtrs* out, int64_t* rejected, int precision, int nthreads) {
    return tab_integrate_adaptive(0, tab, n1, n2, x1_0, d1, x2_0, d2, state_in, n, ctl, max_attempts, st, out, rejected, precision, nthreads);
}

// tab = [10][n2][n1] (reading T6)
int oracle_tabg_integrate_adaptive(const double* tab, int64_t n1, int64_t n2, double x1_0, double d1, double x2_0, double d2,
                                   const double* state_in, int64_t n, const AdaptiveCtl* ctl, int64_t max_attempts,
                                   const StopRule* st, const OutPtrs* out, int64_t* rejected, int precision, int nthreads) {
    return tab_integrate_adaptive(1, tab, n1, n2, x1_0, d1, x2_0, d2, state_in, n, ctl, max_attempts, st, out, rejected, precision, nthreads);
}

}  // extern "C"
