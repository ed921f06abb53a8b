// geo_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, one-particle-at-a-time CPU oracle for the hot path of MALBEC
// (arXiv:1803.08320): fixed-step classical RK4 integration of independent
// null / timelike geodesics in Schwarzschild and Kerr.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call this file.  It shares NO code with the CUDA path
// (paper_1803_08320_b200/csrc/): its own structs, its own algebra.
//
// Algebra used here (chosen to differ from the GPU's 3+1 form):
//   * Schwarzschild: eqs.(29)-(32) of the paper written out literally
//     (PAPER.md:203-211), with p_t(paper) = E (reading G1).
//   * Kerr: Hamilton's equations (3),(4) of
//     H = 1/2 g^{mu nu} p_mu p_nu for the Boyer-Lindquist metric (6)
//     (PAPER.md:73-84), using the separable identity
//       2 rho^2 H = Delta p_r^2 + p_th^2 + (L - a E sin^2 th)^2 / sin^2 th
//                   - [(r^2+a^2) E - a L]^2 / Delta            (p_t = -E, p_phi = L)
//     differentiated by hand.  Pinned (tests/test_oracle_pins.py) against the
//     paper's equatorial eqs.(9)-(12), eqs.(29)-(32) at a=0, high-precision
//     finite differences of H built from metric (6) by matrix inversion, the
//     printed worked example, Tables 1-2, closed forms.
//   * RK4: classical (ref.[19]); autonomous system, step h in tau.
//     State update Kahan-compensated (reading P1) unless flag bit 0.
//   * Stop rules / events / snapshots: DESIGN.md readings B1-B6, S1-S3
//     (PAPER.md:322-327 gives only "final time reached" and "r <= r_+").
//
// Parity-unpinned parts (no closed form exists): finals of escaped / captured
// null rays and eq_cross_r are pinned only by step-halving convergence and the
// long double build of this same file.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared -pthread
//        (oracle/build.py).  -ffp-contract=off: no FMA contraction, so the
//        double build is plain IEEE arithmetic in the written order.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

#include "dp45.h"

namespace {

enum { ORA_SCHWARZSCHILD = 0, ORA_KERR = 1 };
enum { ORA_ST_MAXSTEPS = 0, ORA_ST_CAPTURED = 1, ORA_ST_ESCAPED = 2, ORA_ST_NUMERIC = 3 };
enum { ORA_FLAG_PLAIN_UPDATE = 1,
       ORA_FLAG_CARTESIAN_SNAP = 8 };   // snapshot components r, theta, phi -> x, y, z of eq.(7)

template <class R> struct Hole { int metric; R M, a; };

// State in paper order: y = (t, r, th, phi, p_t=E, p_r, p_th, p_phi=L).
template <class R> struct State { R t, r, th, ph, E, pr, pth, L; };

// ---------------------------------------------------------------------------
// Hamiltonian H = 1/2 g^{mu nu} p_mu p_nu (eq.(4))
// ---------------------------------------------------------------------------
template <class R> R hamiltonian(const Hole<R>& bh, const State<R>& y) {
    const R M = bh.M, a = bh.a;
    const R s = std::sin(y.th), c = std::cos(y.th);
    const R s2 = s * s;
    const R rho2 = y.r * y.r + a * a * c * c;
    const R Delta = y.r * y.r - R(2) * M * y.r + a * a;
    const R P = (y.r * y.r + a * a) * y.E - a * y.L;
    const R Wt = y.L - a * y.E * s2;
    const R N = Delta * y.pr * y.pr + y.pth * y.pth + Wt * Wt / s2 - P * P / Delta;
    return N / (R(2) * rho2);
}

// ---------------------------------------------------------------------------
// Right-hand sides.  out = d/dtau of (t, r, th, phi, p_r, p_th); p_t, p_phi are
// constants of motion (eqs.(13),(32)).
// ---------------------------------------------------------------------------
template <class R> struct Deriv { R t, r, th, ph, pr, pth; };

// eqs.(29)-(32), literally (p_t = E).
template <class R> Deriv<R> rhs_schwarzschild(const Hole<R>& bh, const State<R>& y) {
    const R M = bh.M;
    const R r = y.r;
    const R s = std::sin(y.th), c = std::cos(y.th);
    const R f = R(1) - R(2) * M / r;
    Deriv<R> d;
    d.t = y.E / f;                                               // (29)
    d.r = f * y.pr;                                              // (29)
    d.th = y.pth / (r * r);                                      // (30)
    d.ph = y.L / (r * r * s * s);                                // (30)
    const R g = (-r + R(2) * M);
    d.pr = -M * y.E * y.E / (g * g) - M * y.pr * y.pr / (r * r)  // (31)
           + y.pth * y.pth / (r * r * r) + y.L * y.L / (r * r * r * s * s);
    d.pth = y.L * y.L * c / (r * r * s * s * s);                 // (32)
    return d;
}

// Kerr: separable form, see header.
template <class R> Deriv<R> rhs_kerr(const Hole<R>& bh, const State<R>& y) {
    const R M = bh.M, a = bh.a;
    const R r = y.r, E = y.E, L = y.L;
    const R s = std::sin(y.th), c = std::cos(y.th);
    const R s2 = s * s;
    const R r2a2 = r * r + a * a;
    const R rho2 = r * r + a * a * c * c;
    const R Delta = r * r - R(2) * M * r + a * a;
    const R P = r2a2 * E - a * L;
    const R Wt = L - a * E * s2;
    const R N = Delta * y.pr * y.pr + y.pth * y.pth + Wt * Wt / s2 - P * P / Delta;
    const R twoH = N / rho2;
    Deriv<R> d;
    d.t = (a * Wt + r2a2 * P / Delta) / rho2;                    // -dH/dp_t
    d.r = Delta * y.pr / rho2;                                   // dH/dp_r
    d.th = y.pth / rho2;                                         // dH/dp_th
    d.ph = ((L / s2 - a * E) + a * P / Delta) / rho2;            // dH/dp_phi
    const R dNdr = R(2) * (r - M) * y.pr * y.pr - R(4) * r * E * P / Delta
                   + R(2) * (r - M) * P * P / (Delta * Delta);
    const R dNdth = -R(2) * L * L * c / (s2 * s) + R(2) * a * a * E * E * s * c;
    d.pr = -(dNdr - R(2) * r * twoH) / (R(2) * rho2);            // -dH/dr
    d.pth = -(dNdth + R(2) * a * a * s * c * twoH) / (R(2) * rho2);  // -dH/dth
    return d;
}

template <class R> Deriv<R> rhs(const Hole<R>& bh, const State<R>& y) {
    return bh.metric == ORA_SCHWARZSCHILD ? rhs_schwarzschild(bh, y) : rhs_kerr(bh, y);
}

// ---------------------------------------------------------------------------
// Energy from the mass shell 2L = 2H = -kappa (eq.(5)), future-
// directed root of the quadratic in E obtained from the separable identity:
//   Sigma E^2 - 2 (2 M a r L) E - (Delta W - a^2 L^2) = 0,
//   W = Delta p_r^2 + p_th^2 + L^2/sin^2 th + kappa rho^2.
// ---------------------------------------------------------------------------
template <class R> R energy_from_mass_shell(const Hole<R>& bh, R r, R th, R pr, R pth, R L, R kappa) {
    const R M = bh.M, a = bh.a;
    const R s = std::sin(th), c = std::cos(th);
    const R s2 = s * s;
    const R rho2 = r * r + a * a * c * c;
    const R Delta = r * r - R(2) * M * r + a * a;
    const R Sigma = (r * r + a * a) * (r * r + a * a) - a * a * Delta * s2;
    const R W = Delta * pr * pr + pth * pth + L * L / s2 + kappa * rho2;
    const R b = R(2) * M * a * r * L;
    const R disc = b * b + Sigma * (Delta * W - a * a * L * L);
    return (b + std::sqrt(disc)) / Sigma;
}

// ---------------------------------------------------------------------------
// One particle: init, RK4 loop, stop rules, events, snapshots, final record.
// ---------------------------------------------------------------------------
struct StopRule { double r_capture, r_escape; int32_t kind; int32_t flags; };

struct OutPtrs {
    double* final_state;    // [8][n]   t, r, th, phi, p_t(=E), p_r, p_th, p_phi
    int32_t* status;        // [n]
    int64_t* steps_done;    // [n]
    double* eq_cross_r;     // [n] or null
    double* health;         // [n] or null
    double* snapshots;      // [n][snap_capacity][ncomp] or null
    int64_t snap_capacity;
    uint32_t snap_mask;
    int32_t* snap_count;    // [n] or null
};

template <class R> bool finite6(const State<R>& y) {
    return std::isfinite(y.t) && std::isfinite(y.r) && std::isfinite(y.th) &&
           std::isfinite(y.ph) && std::isfinite(y.pr) && std::isfinite(y.pth);
}

template <class R> R component(const State<R>& y, int k) {
    switch (k) {
        case 0: return y.t;  case 1: return y.r;  case 2: return y.th;  case 3: return y.ph;
        case 4: return y.E;  case 5: return y.pr; case 6: return y.pth; default: return y.L;
    }
}

template <class R> State<R> shifted(const State<R>& y, R w, const Deriv<R>& k) {
    State<R> z = y;               // E, L unchanged (eqs.(13),(32))
    z.t = y.t + w * k.t;
    z.r = y.r + w * k.r;
    z.th = y.th + w * k.th;
    z.ph = y.ph + w * k.ph;
    z.pr = y.pr + w * k.pr;
    z.pth = y.pth + w * k.pth;
    return z;
}

// y <- y + delta, Kahan-compensated with carried error term c (reading P1).
template <class R> void kahan_add(R& y, R& c, R delta, bool plain) {
    if (plain) { y = y + delta; return; }
    const R yk = delta - c;
    const R tsum = y + yk;
    c = (tsum - y) - yk;
    y = tsum;
}

// Boyer-Lindquist -> Cartesian, eq.(7) PAPER.md:88-93 (the paper's output format):
//   x = sqrt(r^2 + a^2) sin(th) cos(ph),  y = sqrt(r^2 + a^2) sin(th) sin(ph),  z = r cos(th).
template <class R> void cartesian_eq7(R a, const State<R>& y, R& X, R& Y, R& Z) {
    const R w = std::sqrt(y.r * y.r + a * a);
    X = w * std::sin(y.th) * std::cos(y.ph);
    Y = w * std::sin(y.th) * std::sin(y.ph);
    Z = y.r * std::cos(y.th);
}

template <class R>
void write_snapshot(const OutPtrs& o, int64_t i, int64_t slot, const State<R>& y, R a, bool cartesian) {
    if (!o.snapshots || slot >= o.snap_capacity) return;   // S3: drop, never overflow
    int ncomp = 0;
    for (int k = 0; k < 8; ++k) ncomp += (o.snap_mask >> k) & 1u;
    double* dst = o.snapshots + (i * o.snap_capacity + slot) * ncomp;
    R xyz[3] = {y.r, y.th, y.ph};
    if (cartesian) cartesian_eq7(a, y, xyz[0], xyz[1], xyz[2]);
    int j = 0;
    for (int k = 0; k < 8; ++k)
        if ((o.snap_mask >> k) & 1u) dst[j++] = (double)((k >= 1 && k <= 3) ? xyz[k - 1] : component(y, k));
}

template <class R>
void integrate_one(const Hole<R>& bh, const double* state_in, int64_t n, int64_t i, R h,
                   int64_t nsteps, const StopRule& st, int64_t snapshot_every, const OutPtrs& o) {
    const R kappa = st.kind == 0 ? R(1) : R(0);
    const bool plain = (st.flags & ORA_FLAG_PLAIN_UPDATE) != 0;
    const bool cart = (st.flags & ORA_FLAG_CARTESIAN_SNAP) != 0;
    const R rc = (R)st.r_capture, re = (R)st.r_escape;
    const R half_pi = (R)1.5707963267948966;          // nearest double to pi/2 (reading B5)

    State<R> y;
    y.t = R(0);
    y.r = (R)state_in[0 * n + i];
    y.th = (R)state_in[1 * n + i];
    y.ph = (R)state_in[2 * n + i];
    y.pr = (R)state_in[3 * n + i];
    y.pth = (R)state_in[4 * n + i];
    y.L = (R)state_in[5 * n + i];
    y.E = energy_from_mass_shell(bh, y.r, y.th, y.pr, y.pth, y.L, kappa);
    R ct = 0, cr = 0, cth = 0, cph = 0, cpr = 0, cpth = 0;   // Kahan error terms

    int32_t status = -1;
    int64_t steps = 0;
    int64_t snaps = 0;
    R eq_cross = std::numeric_limits<R>::quiet_NaN();
    bool crossed = false;

    // B1: tests on y0 before the first step.
    if (!(y.r >= rc)) status = ORA_ST_CAPTURED;
    else if (!finite6(y) || !std::isfinite(y.E)) status = ORA_ST_NUMERIC;
    else {
        if (snapshot_every > 0) { write_snapshot(o, i, 0, y, bh.a, cart); snaps = 1; }   // S1: slot 0 = y0
        if (y.r > re) status = ORA_ST_ESCAPED;
        else if (nsteps == 0) status = ORA_ST_MAXSTEPS;
    }

    while (status < 0) {
        // classical RK4; B2: guard every evaluation point.
        const Deriv<R> k1 = rhs(bh, y);
        const State<R> y2 = shifted(y, h / R(2), k1);
        if (!(y2.r >= rc)) { status = ORA_ST_CAPTURED; break; }
        const Deriv<R> k2 = rhs(bh, y2);
        const State<R> y3 = shifted(y, h / R(2), k2);
        if (!(y3.r >= rc)) { status = ORA_ST_CAPTURED; break; }
        const Deriv<R> k3 = rhs(bh, y3);
        const State<R> y4 = shifted(y, h, k3);
        if (!(y4.r >= rc)) { status = ORA_ST_CAPTURED; break; }
        const Deriv<R> k4 = rhs(bh, y4);

        State<R> yn = y;
        R nt = ct, nr = cr, nth = cth, nph = cph, npr = cpr, npth = cpth;
        const R w = h / R(6);
        kahan_add(yn.t, nt, w * (k1.t + R(2) * k2.t + R(2) * k3.t + k4.t), plain);
        kahan_add(yn.r, nr, w * (k1.r + R(2) * k2.r + R(2) * k3.r + k4.r), plain);
        kahan_add(yn.th, nth, w * (k1.th + R(2) * k2.th + R(2) * k3.th + k4.th), plain);
        kahan_add(yn.ph, nph, w * (k1.ph + R(2) * k2.ph + R(2) * k3.ph + k4.ph), plain);
        kahan_add(yn.pr, npr, w * (k1.pr + R(2) * k2.pr + R(2) * k3.pr + k4.pr), plain);
        kahan_add(yn.pth, npth, w * (k1.pth + R(2) * k2.pth + R(2) * k3.pth + k4.pth), plain);

        if (!(yn.r >= rc)) { status = ORA_ST_CAPTURED; break; }     // B2: end point
        if (!finite6(yn)) { status = ORA_ST_NUMERIC; break; }       // B6

        // accept the step
        if (!crossed) {                                             // B5
            const R d0 = y.th - half_pi, d1 = yn.th - half_pi;
            if (d0 * d1 < R(0)) {
                crossed = true;
                eq_cross = y.r + (yn.r - y.r) * (half_pi - y.th) / (yn.th - y.th);
            }
        }
        y = yn; ct = nt; cr = nr; cth = nth; cph = nph; cpr = npr; cpth = npth;
        ++steps;
        if (snapshot_every > 0 && steps % snapshot_every == 0) {    // S1
            write_snapshot(o, i, snaps, y, bh.a, cart);
            ++snaps;
        }
        if (y.r > re) status = ORA_ST_ESCAPED;                      // B3
        else if (steps >= nsteps) status = ORA_ST_MAXSTEPS;         // B4
    }

    for (int k = 0; k < 8; ++k) o.final_state[(int64_t)k * n + i] = (double)component(y, k);
    o.status[i] = status;
    o.steps_done[i] = steps;
    if (o.eq_cross_r) o.eq_cross_r[i] = (double)eq_cross;
    if (o.health) o.health[i] = (double)std::fabs(R(2) * hamiltonian(bh, y) + kappa);   // B7
    if (o.snap_count) o.snap_count[i] = (int32_t)snaps;
}

template <class R>
void integrate_range(int metric, double M, double a, const double* state_in, int64_t n,
                     int64_t lo, int64_t hi, double h, int64_t nsteps, const StopRule& st,
                     int64_t snapshot_every, const OutPtrs& o) {
    Hole<R> bh{metric, (R)M, (R)a};
    for (int64_t i = lo; i < hi; ++i)
        integrate_one<R>(bh, state_in, n, i, (R)h, nsteps, st, snapshot_every, o);
}

// ---------------------------------------------------------------------------
// adaptive embedded Runge-Kutta 5(4) ("others method of the RK family will be included
// soon").  The pair is Dormand & Prince's (J. Comput. Appl. Math. 6 (1980) 19, table 2 --
// the DOPRI5 of Hairer, Norsett & Wanner, ref.[19] of the paper): 7 stages, first-same-as-last, the
// 5th-order solution is propagated (local extrapolation), the difference to the embedded 4th-order
// solution estimates the local error.  Step control, the textbook elementary controller:
//   err = max_c |e_c| / (atol + rtol * max(|y_c|, |ynew_c|))  over the 6 evolving components,
//   accept iff err <= 1,   h <- h * min(5, max(0.2, 0.9 * err^(-1/5))),  after a rejection never > 1.
// "The final evolution time is reached": with a finite tau_end the step that would pass it
// is shortened to land on it (when tau + 1.01 h >= tau_end) and the particle ends with MAXSTEPS.
// Stop rules as for RK4 (readings B1-B5): capture guard on every stage point and the end point (the
// attempt is not taken), escape test after an accepted step, `nsteps` caps the ATTEMPTS.
// ---------------------------------------------------------------------------
template <class R> R comp6(const State<R>& y, int c) {
    switch (c) { case 0: return y.t; case 1: return y.r; case 2: return y.th; case 3: return y.ph;
                 case 4: return y.pr; default: return y.pth; }
}
template <class R> R dcomp6(const Deriv<R>& k, int c) {
    switch (c) { case 0: return k.t; case 1: return k.r; case 2: return k.th; case 3: return k.ph;
                 case 4: return k.pr; default: return k.pth; }
}
template <class R> void set6(State<R>& y, int c, R v) {
    switch (c) { case 0: y.t = v; break; case 1: y.r = v; break; case 2: y.th = v; break;
                 case 3: y.ph = v; break; case 4: y.pr = v; break; default: y.pth = v; }
}

template <class R>
void integrate_one_adaptive(const Hole<R>& bh, const double* state_in, int64_t n, int64_t i,
                            const AdaptiveCtl& ctl, int64_t max_attempts, const StopRule& st,
                            const OutPtrs& o, int64_t* rejected_out) {
    static const DP45 T;
    const R kappa = st.kind == 0 ? R(1) : R(0);
    const R rc = (R)st.r_capture, re = (R)st.r_escape;
    const R half_pi = (R)1.5707963267948966;
    State<R> y;
    y.t = R(0);
    y.r = (R)state_in[0 * n + i];
    y.th = (R)state_in[1 * n + i];
    y.ph = (R)state_in[2 * n + i];
    y.pr = (R)state_in[3 * n + i];
    y.pth = (R)state_in[4 * n + i];
    y.L = (R)state_in[5 * n + i];
    y.E = energy_from_mass_shell(bh, y.r, y.th, y.pr, y.pth, y.L, kappa);
    R cc[6] = {0, 0, 0, 0, 0, 0};                     // Kahan error terms (reading P1)
    R h = (R)ctl.h0;
    R tau = R(0);
    const R tau_end = (R)ctl.tau_end;
    const bool dense = ctl.snap_dtau > 0.0 && o.snapshots != nullptr;   // reading A3: records at tau_j = j * snap_dtau
    const bool cart = (st.flags & ORA_FLAG_CARTESIAN_SNAP) != 0;
    const R dtau = (R)ctl.snap_dtau;
    int64_t next_j = 0;                               // records produced so far = index of the next one
    int32_t status = -1;
    int64_t steps = 0, attempts = 0, rejected = 0;
    R eq_cross = std::numeric_limits<R>::quiet_NaN();
    bool crossed = false;

    if (!(y.r >= rc)) status = ORA_ST_CAPTURED;                      // B1
    else if (!finite6(y) || !std::isfinite(y.E)) status = ORA_ST_NUMERIC;
    else {
        if (dense) { write_snapshot(o, i, 0, y, bh.a, cart); next_j = 1; }   // record 0 = y0 (tau = 0), as S1
        if (y.r > re) status = ORA_ST_ESCAPED;
        else if (max_attempts == 0) status = ORA_ST_MAXSTEPS;
    }

    Deriv<R> k[DP45::S];
    if (status < 0) k[0] = rhs(bh, y);
    while (status < 0) {
        const bool last = tau + R(1.01) * h >= tau_end;             // land on the final time
        if (last) h = tau_end - tau;
        bool captured = false;
        for (int s = 1; s < DP45::S - 1; ++s) {                      // stages 2..6
            State<R> ys = y;
            for (int c = 0; c < 6; ++c) {
                R acc = R(0);
                for (int j = 0; j < s; ++j) acc += (R)T.a[s][j] * dcomp6(k[j], c);
                set6(ys, c, comp6(y, c) + h * acc);
            }
            if (!(ys.r >= rc)) { captured = true; break; }           // B2 on every evaluation point
            k[s] = rhs(bh, ys);
        }
        ++attempts;
        if (captured) { status = ORA_ST_CAPTURED; break; }
        // 5th-order solution (compensated update, committed only on acceptance); stage 7 sits on it
        State<R> yn = y;
        R cn[6];
        for (int c = 0; c < 6; ++c) {
            R acc5 = R(0);
            for (int j = 0; j < DP45::S - 1; ++j) acc5 += (R)T.a[6][j] * dcomp6(k[j], c);
            R v = comp6(y, c);
            cn[c] = cc[c];
            kahan_add(v, cn[c], h * acc5, false);
            set6(yn, c, v);
        }
        if (!(yn.r >= rc)) { status = ORA_ST_CAPTURED; break; }      // B2: end point
        const bool fin = finite6(yn);
        R err = R(0);
        if (fin) {
            k[6] = rhs(bh, yn);
            for (int c = 0; c < 6; ++c) {
                R acce = R(0);                                       // (b5 - b4) . k, b5_7 = 0
                for (int j = 0; j < DP45::S; ++j)
                    acce += ((R)(j < 6 ? T.a[6][j] : 0.0L) - (R)T.b4[j]) * dcomp6(k[j], c);
                const R sc = (R)ctl.atol + (R)ctl.rtol * std::max(std::fabs(comp6(y, c)), std::fabs(comp6(yn, c)));
                const R ec = std::fabs(h * acce) / sc;
                if (!(ec <= err)) err = ec;                          // max; a NaN sticks
            }
        }
        if (fin && std::isinf(ctl.rtol)) err = R(0);                 // fixed-step mode: no error test
        R fac = err > R(0) ? R(0.9) * std::pow(err, R(-0.2)) : (err == R(0) ? R(5) : R(0.2));   // NaN estimate: shrink
        if (!(fac >= R(0.2))) fac = R(0.2);
        if (fac > R(5)) fac = R(5);
        if (std::isinf(ctl.rtol)) fac = R(1);                        // rtol = +inf: fixed step h0 (order tests)
        if (!fin || !(err <= R(1))) {                                // reject
            ++rejected;
            h *= std::min(fac, R(1));
            // reading A2: a rejected step below h_min ends with NUMERIC; so does a non-finite attempt in fixed-step
            // mode (the same step would be retried forever) and a step size that has underflowed to zero
            if ((std::isinf(ctl.rtol) && !fin) || !(std::fabs(h) >= (R)ctl.h_min) || !(std::fabs(h) > R(0))) {
                status = ORA_ST_NUMERIC; break;
            }
            if (attempts >= max_attempts) { status = ORA_ST_MAXSTEPS; break; }
            continue;
        }
        if (!crossed) {                                              // B5
            const R d0 = y.th - half_pi, d1 = yn.th - half_pi;
            if (d0 * d1 < R(0)) {
                crossed = true;
                eq_cross = y.r + (yn.r - y.r) * (half_pi - y.th) / (yn.th - y.th);
            }
        }
        const R tau_new = last ? tau_end : tau + h;                  // the final time is landed on exactly
        if (dense) {                                                 // A3: every record time in (tau, tau_new]
            for (;;) {
                const R tj = (R)next_j * dtau;
                if (!(tj <= tau_new)) break;
                R w[7];
                dp45_dense_weights<R>((tj - tau) / h, w);
                State<R> ys = y;
                for (int c = 0; c < 6; ++c) {
                    R acc = R(0);
                    for (int j = 0; j < DP45::S; ++j) acc += w[j] * dcomp6(k[j], c);
                    set6(ys, c, comp6(y, c) + h * acc);
                }
                write_snapshot(o, i, next_j, ys, bh.a, cart);
                ++next_j;
            }
        }
        y = yn;
        for (int c = 0; c < 6; ++c) cc[c] = cn[c];
        k[0] = k[6];                                                 // first same as last
        ++steps;
        tau = tau_new;
        h *= fac;
        if (y.r > re) status = ORA_ST_ESCAPED;                       // B3
        else if (last || attempts >= max_attempts) status = ORA_ST_MAXSTEPS;   // final time / B4 (cap on attempts)
    }
    for (int q = 0; q < 8; ++q) o.final_state[(int64_t)q * n + i] = (double)component(y, q);
    o.status[i] = status;
    o.steps_done[i] = steps;
    if (o.eq_cross_r) o.eq_cross_r[i] = (double)eq_cross;
    if (o.health) o.health[i] = (double)std::fabs(R(2) * hamiltonian(bh, y) + kappa);
    if (dense && o.snap_count) o.snap_count[i] = (int32_t)next_j;
    if (rejected_out) rejected_out[i] = rejected;
}

}  // namespace

extern "C" {

// Returns 0 on success, 1 on invalid arguments.  All pointers are HOST memory.
// precision: 0 = double, 1 = long double (x87 80-bit).  nthreads: particle-
// parallel outer loop only (contiguous chunks); per-particle arithmetic does
// not depend on it.
int oracle_integrate(int metric, double M, double a, const double* state_in, int64_t n, double h,
                     int64_t nsteps, const StopRule* stop, int64_t snapshot_every,
                     const OutPtrs* out, int precision, int nthreads) {
    if (!stop || !out || n < 0 || nsteps < 0 || snapshot_every < 0) return 1;
    if (!(M > 0) || !(std::fabs(a) <= M) || !std::isfinite(h) || h == 0.0) return 1;
    if (metric != ORA_SCHWARZSCHILD && metric != ORA_KERR) return 1;
    if (metric == ORA_SCHWARZSCHILD && a != 0.0) return 1;
    if (n == 0) return 0;
    if (!state_in || !out->final_state || !out->status || !out->steps_done) return 1;
    if (snapshot_every > 0 && (!out->snapshots || !out->snap_count || out->snap_capacity < 1 ||
                               (out->snap_mask & 0xFFu) == 0)) return 1;
    if (nthreads < 1) nthreads = 1;
    if ((int64_t)nthreads > n) nthreads = (int)n;
    auto run = [&](int64_t lo, int64_t hi) {
        if (precision == 1)
            integrate_range<long double>(metric, M, a, state_in, n, lo, hi, h, nsteps, *stop, snapshot_every, *out);
        else
            integrate_range<double>(metric, M, a, state_in, n, lo, hi, h, nsteps, *stop, snapshot_every, *out);
    };
    if (nthreads == 1) { run(0, n); return 0; }
    std::vector<std::thread> pool;
    // interleaved small blocks so captured/escaped mixes balance across threads
    const int64_t block = 64;
    const int64_t nblocks = (n + block - 1) / block;
    for (int t = 0; t < nthreads; ++t)
        pool.emplace_back([&, t]() {
            for (int64_t b = t; b < nblocks; b += nthreads)
                run(b * block, std::min<int64_t>(n, (b + 1) * block));
        });
    for (auto& th : pool) th.join();
    return 0;
}

// Adaptive RK5(4).  ctl = {h0, rtol, atol, h_min}; max_attempts caps accepted + rejected
// attempts per particle; rejected: [n] or NULL.  ctl->snap_dtau > 0: dense-output records into out->snapshots (reading A3).
int oracle_integrate_adaptive(int metric, double M, double a, const double* state_in, int64_t n,
                              const AdaptiveCtl* ctl, int64_t max_attempts, const StopRule* stop,
                              const OutPtrs* out, int64_t* rejected, int precision, int nthreads) {
    if (!stop || !out || !ctl || n < 0 || max_attempts < 0) return 1;
    if (!(M > 0) || !(std::fabs(a) <= M)) return 1;
    if (!std::isfinite(ctl->h0) || !(ctl->h0 > 0.0) || !(ctl->rtol >= 0) || !(ctl->atol >= 0) ||
        !(ctl->rtol + ctl->atol > 0) || !(ctl->h_min >= 0) || !(ctl->tau_end > 0) || !(ctl->snap_dtau >= 0)) return 1;
    if (ctl->snap_dtau > 0 && (!out->snapshots || !out->snap_count || out->snap_capacity < 1 || (out->snap_mask & 0xFFu) == 0)) return 1;
    if (metric != ORA_SCHWARZSCHILD && metric != ORA_KERR) return 1;
    if (metric == ORA_SCHWARZSCHILD && a != 0.0) return 1;
    if (n == 0) return 0;
    if (!state_in || !out->final_state || !out->status || !out->steps_done) return 1;
    if (nthreads < 1) nthreads = 1;
    if ((int64_t)nthreads > n) nthreads = (int)n;
    auto run = [&](int64_t lo, int64_t hi) {
        for (int64_t i = lo; i < hi; ++i) {
            if (precision == 1) {
                Hole<long double> bh{metric, (long double)M, (long double)a};
                integrate_one_adaptive<long double>(bh, state_in, n, i, *ctl, max_attempts, *stop, *out, rejected);
            } else {
                Hole<double> bh{metric, M, a};
                integrate_one_adaptive<double>(bh, state_in, n, i, *ctl, max_attempts, *stop, *out, rejected);
            }
        }
    };
    if (nthreads == 1) { run(0, n); return 0; }
    std::vector<std::thread> pool;
    const int64_t block = 64;
    const int64_t nblocks = (n + block - 1) / block;
    for (int t = 0; t < nthreads; ++t)
        pool.emplace_back([&, t]() {
            for (int64_t b = t; b < nblocks; b += nthreads)
                run(b * block, std::min<int64_t>(n, (b + 1) * block));
        });
    for (auto& th : pool) th.join();
    return 0;
}

// w_i(theta), i = 1..7, of the dense output (reading A3), as doubles.
void oracle_dp45_dense_weights(double theta, double* w7) {
    long double w[7];
    dp45_dense_weights<long double>((long double)theta, w);
    for (int i = 0; i < 7; ++i) w7[i] = (double)w[i];
}

// The Butcher tableau the adaptive path uses, as doubles: c[7], a[7][7] (row-major), b5[7], b4[7].
void oracle_dp45_tableau(double* c, double* a, double* b5, double* b4) {
    static const DP45 T;
    for (int i = 0; i < 7; ++i) {
        c[i] = (double)T.c[i];
        b5[i] = (double)(i < 6 ? T.a[6][i] : 0.0L);
        b4[i] = (double)T.b4[i];
        for (int j = 0; j < 7; ++j) a[7 * i + j] = (double)(j < i ? T.a[i][j] : 0.0L);
    }
}

// d/dtau of (t, r, th, phi, p_r, p_th) at y = (t, r, th, phi, E, p_r, p_th, L).
void oracle_rhs(int metric, double M, double a, const double* y8, double* d6, int precision) {
    if (precision == 1) {
        Hole<long double> bh{metric, M, a};
        State<long double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
        Deriv<long double> d = rhs(bh, y);
        d6[0] = (double)d.t; d6[1] = (double)d.r; d6[2] = (double)d.th;
        d6[3] = (double)d.ph; d6[4] = (double)d.pr; d6[5] = (double)d.pth;
    } else {
        Hole<double> bh{metric, M, a};
        State<double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
        Deriv<double> d = rhs(bh, y);
        d6[0] = d.t; d6[1] = d.r; d6[2] = d.th; d6[3] = d.ph; d6[4] = d.pr; d6[5] = d.pth;
    }
}

double oracle_hamiltonian(double M, double a, const double* y8) {
    Hole<double> bh{ORA_KERR, M, a};
    State<double> y{y8[0], y8[1], y8[2], y8[3], y8[4], y8[5], y8[6], y8[7]};
    return hamiltonian(bh, y);
}

double oracle_energy(double M, double a, double r, double th, double pr, double pth, double L, double kappa) {
    Hole<double> bh{ORA_KERR, M, a};
    return energy_from_mass_shell<double>(bh, r, th, pr, pth, L, kappa);
}

}  // extern "C"
