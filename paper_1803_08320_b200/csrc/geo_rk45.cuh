// geo_rk45.cuh -- adaptive embedded Runge-Kutta 5(4) stepper ("others method of the RK
// family will be included soon"), one persistent kernel on the same 3+1 RHS, work queue and
// stop rules as the fixed-step RK4 kernel of geo_kernel.cuh.
//
// Pair: Dormand & Prince 5(4) with 7 stages, first-same-as-last (DOPRI5 of ref.[19] of the paper); the
// 5th-order solution is propagated, its difference to the embedded 4th-order solution estimates the local
// error.  Per-geodesic step control (elementary controller):
//     err = max_c |e_c| / (atol + rtol max(|y_c|, |ynew_c|))   over the 6 evolving components,
//     accept iff err <= 1,   h <- h min(5, max(0.2, 0.9 err^(-1/5)))   (never enlarged after a rejection),
// rtol = +inf: fixed step h0.  Stop rules: capture guard on every stage point and on the end point (that
// attempt is not taken), escape after an accepted step, a finite tau_end is landed on ("the final evolution
// time is reached"), max_attempts caps accepted + rejected attempts.
// Step counts differ by orders of magnitude between rays (far field vs. near the hole), so the work queue
// of DESIGN.md A5 is what keeps the lanes busy here.
#pragma once
#include "geo_kernel.cuh"
#include "geo_tab.cuh"
#include "geo_tabg.cuh"
#ifndef GEO_RK45_CTAS
#define GEO_RK45_CTAS 3      // resident CTAs per SM the kernel is compiled for (168 registers, no spills)
#endif

namespace geo {

struct AdaptiveParams {
    const double* in;   // [6][n]
    long long n;
    double h0, rtol, atol, h_min, tau_end;
    int fixed_step;     // rtol == +inf
    int max_attempts;
    double r_capture, r_escape, kappa;
    double* fin;        // [8][n]
    int* status;
    long long* steps_done;
    double* eq_cross_r;
    double* health;
    int* rejected;      // [n] or null
    unsigned long long* counter;
    // dense output (reading A3): records at tau_j = j * snap_dtau from the pair's continuous extension
    double snap_dtau;   // 0: none
    double* snaps;      // [n][snap_cap][ncomp]
    long long snap_cap;
    unsigned snap_mask;
    int ncomp;
    int cartesian;
    int* snap_count;
    Hole bh;
    TabMetric tm;       // METRIC_TAB: the five-field table (reading T7)
    TabgMetric tgm;     // METRIC_TABG: the ten-field table (readings T6 + T7)
};

enum { METRIC_SCHW = 0, METRIC_KERR = 1, METRIC_TAB = 2, METRIC_TABG = 3 };
__host__ __device__ constexpr bool metric_is_tab(int m) { return m == METRIC_TAB || m == METRIC_TABG; }

// Butcher tableau (Dormand & Prince 1980, table 2).  e = b5 - b4.
namespace dp {
constexpr double a21 = 1.0 / 5;
constexpr double a31 = 3.0 / 40, a32 = 9.0 / 40;
constexpr double a41 = 44.0 / 45, a42 = -56.0 / 15, a43 = 32.0 / 9;
constexpr double a51 = 19372.0 / 6561, a52 = -25360.0 / 2187, a53 = 64448.0 / 6561, a54 = -212.0 / 729;
constexpr double a61 = 9017.0 / 3168, a62 = -355.0 / 33, a63 = 46732.0 / 5247, a64 = 49.0 / 176, a65 = -5103.0 / 18656;
constexpr double b1 = 35.0 / 384, b3 = 500.0 / 1113, b4 = 125.0 / 192, b5 = -2187.0 / 6784, b6 = 11.0 / 84;
// dense output (Hairer's dopri5, "contd5"): coefficients of the fifth interpolation term
constexpr double d1 = -12715105075.0 / 11282082432.0, d3 = 87487479700.0 / 32700410799.0, d4 = -10690763975.0 / 1880347072.0,
                 d5 = 701980252875.0 / 199316789632.0, d6 = -1453857185.0 / 822651844.0, d7 = 69997945.0 / 29380423.0;
constexpr double e1 = 35.0 / 384 - 5179.0 / 57600, e3 = 500.0 / 1113 - 7571.0 / 16695, e4 = 125.0 / 192 - 393.0 / 640,
                 e5 = -2187.0 / 6784 + 92097.0 / 339200, e6 = 11.0 / 84 - 187.0 / 2100, e7 = -1.0 / 40;
}  // namespace dp

// x^(-1/5) for the step-size controller: single-precision seed (MUFU lg2/ex2), two Newton steps on y^-5 = x
// (y <- y (6 - x y^5)/5, relative error 3 eps^2 per step), a few ulp in all.  The controller clamps the factor to
// [0.2, 5], i.e. only x in [1.9e-4, 1.8e3] matters: x is clamped to [1e-5, 1e4] first, which keeps the float seed
// in range (+inf included).  Replaces pow(x, -0.2) (~150 instructions with its special-case paths).
__device__ __forceinline__ double inv_fifth_root(double x) {
    const double xc = fmin(fmax(x, 1.0e-5), 1.0e4);
    double y = (double)exp2f(-0.2f * __log2f((float)xc));
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double y2 = y * y;
        const double y5 = y2 * y2 * y;
        y *= fma(-0.2 * xc, y5, 1.2);
    }
    return y;
}

// |e| / sc with one faithfully rounded reciprocal instead of an IEEE division (the quotient may differ from the
// oracle's by an ulp -- like every FMA-contracted sum that feeds it)
__device__ __forceinline__ double scaled_err(double e, double sc) { return fabs(e) * rcp_nr(sc); }

// the four components that feed back into the RHS
struct K4 {
    double r, th, pr, pth;
};

template <bool KERR>
__device__ __forceinline__ void rhs_at(const Hole& bh, double r, double th, double pr, double pth, double E, double L,
                                       Deriv& d) {
    double s2, sc;
    sin2_sincos(bh.tc, th, s2, sc);
    rhs<KERR>(bh, r, s2, sc, pr, pth, E, L, d);
}

__device__ __forceinline__ K4 k4_of(const Deriv& d) { return K4{d.r, d.th, d.pr, d.pth}; }

// T7: one evaluation of the tabulated right-hand side (gathered stencil), out of line -- the attempt has seven of them and
// an unrolled copy each would be ~2300 instructions of evaluator.  Returns false outside the table's domain.
__device__ __noinline__ bool tab_eval(const TabMetric& m, double x1, double x2, double p1, double p2, double E, double L, Deriv* d) {
    TabFields F;
    const bool in = tab_fields(m, x1, x2, F);
    TabDeriv td;
    tab_rhs(F, p1, p2, E, L, td);
    d->t = td.t; d->r = td.x1; d->th = td.x2; d->ph = td.ph; d->pr = td.p1; d->pth = td.p2;
    return in;
}

// T6 + T7: the same for the ten-field table (gathered stencil; the per-lane stencil cache of geo_tabg_rk4_kernel is not used
// here: an adaptive step moves across cells).
__device__ __noinline__ bool tabg_eval(const TabgMetric& m, double x1, double x2, double p1, double p2, double E, double L, Deriv* d) {
    TabgFields F;
    const bool in = tabg_fields(m, x1, x2, F);
    TabDeriv td;
    tabg_rhs(F, p1, p2, E, L, td);
    d->t = td.t; d->r = td.x1; d->th = td.x2; d->ph = td.ph; d->pr = td.p1; d->pth = td.p2;
    return in;
}

// right-hand side of the selected metric at one evaluation point; false: outside the domain (tabulated metric only)
template <int METRIC>
__device__ __forceinline__ bool rhs_metric(const AdaptiveParams& p, double r, double th, double pr, double pth, double E, double L, Deriv& d) {
    if (METRIC == METRIC_TAB) return tab_eval(p.tm, r, th, pr, pth, E, L, &d);
    if (METRIC == METRIC_TABG) return tabg_eval(p.tgm, r, th, pr, pth, E, L, &d);
    rhs_at<METRIC == METRIC_KERR>(p.bh, r, th, pr, pth, E, L, d);
    return true;
}

// One component of the continuous extension at theta in [0, 1] (reading A3), nested as in dopri5's contd5:
//   y + theta (r2 + theta1 (r3 + theta (r4 + theta1 r5))),  r2 = ynew - y, r3 = h k1 - r2, r4 = r2 - h k7 - r3, r5 = h sum d_i k_i
__device__ __forceinline__ double contd5(double theta, double y, double ynew, double hk1, double hk7, double hdk) {
    const double th1 = 1.0 - theta;
    const double r2 = ynew - y, r3 = hk1 - r2, r4 = r2 - hk7 - r3;
    return fma(theta, fma(th1, fma(theta, fma(th1, hdk, r4), r3), r2), y);
}

// DENSE: dense-output records (geo_adaptive.snap_dtau > 0); a separate instantiation so that the plain kernel keeps its
// register budget.
template <int METRIC, bool DENSE>
__global__ void __launch_bounds__(kBlock, (DENSE || metric_is_tab(METRIC)) ? 2 : GEO_RK45_CTAS) geo_rk45_kernel(const __grid_constant__ AdaptiveParams p) {
    constexpr bool kTab = metric_is_tab(METRIC);      // a tabulated metric: domain tests (T4, T7), E undefined until y0 is inside
    const unsigned lane = threadIdx.x & 31u;
    const Hole& bh = p.bh;
    long long idx = -1;
    bool active = false, exhausted = false;
    double t = 0, r = 0, th = 0, ph = 0, pr = 0, pth = 0, E = 0, L = 0;
    double ct = 0, cr = 0, cth = 0, cph = 0, cpr = 0, cpth = 0;     // Kahan error terms (reading P1)
    double h = p.h0, tau = 0;
    Deriv k1;                                                        // f(y): first same as last
    k1.t = k1.r = k1.th = k1.ph = k1.pr = k1.pth = 0;
    int steps = 0, attempts = 0, rejected = 0;
    double eqc = 0;
    bool crossed = false;
    int next_j = 0;                                                  // DENSE: records produced = index of the next one

    // DENSE: one record (paper order; components 1..3 optionally Cartesian, eq.(7)) into slot j of this particle
    auto write_record = [&](int j, double rt, double rr, double rth, double rph, double rpr, double rpth) {
        if (j < p.snap_cap) {                                        // S3: drop beyond capacity, keep counting
            double c1 = rr, c2 = rth, c3 = rph;
            if (p.cartesian) cartesian_eq7(bh.tc, bh.a2, rr, rth, rph, c1, c2, c3);
            double* dst = p.snaps + ((size_t)idx * (size_t)p.snap_cap + (size_t)j) * p.ncomp;
            store_record_global(dst, p.snap_mask, rt, c1, c2, c3, E, rpr, rpth, L);
        }
    };

    auto finish = [&](int st) {
        long long n = p.n;
        asm volatile("" : "+l"(n));
        p.fin[0 * n + idx] = t;
        p.fin[1 * n + idx] = r;
        p.fin[2 * n + idx] = th;
        p.fin[3 * n + idx] = ph;
        p.fin[4 * n + idx] = E;
        p.fin[5 * n + idx] = pr;
        p.fin[6 * n + idx] = pth;
        p.fin[7 * n + idx] = L;
        p.status[idx] = st;
        p.steps_done[idx] = (long long)steps;
        if (p.eq_cross_r) p.eq_cross_r[idx] = crossed ? eqc : __longlong_as_double(0x7ff8000000000000LL);
        if (p.health) {
            if (METRIC == METRIC_TABG) {
                TabgFields F;
                double hv = __longlong_as_double(0x7ff8000000000000LL);
                if (tabg_fields_cold(p.tgm, r, th, F) && (__double2hiint(E) & 0x7ff00000) != 0x7ff00000) {
                    const TabgAux A = tabg_aux(F.v, pr, pth, L, E);
                    hv = fabs(-(A.W * A.W) / (F.v[0] * F.v[0]) + A.gpp + p.kappa);
                }
                p.health[idx] = hv;
            } else if (METRIC == METRIC_TAB) {
                TabFields F;
                double hv = __longlong_as_double(0x7ff8000000000000LL);
                if (tab_fields_cold(p.tm, r, th, F) && (__double2hiint(E) & 0x7ff00000) != 0x7ff00000) {
                    const double W = fma(F.be, L, E);
                    hv = fabs(-(W * W) / (F.al * F.al) + pr * pr / F.g11 + pth * pth / F.g22 + L * L / F.g33 + p.kappa);
                }
                p.health[idx] = hv;
            } else {
                p.health[idx] = health_3p1(bh, r, th, pr, pth, E, L, p.kappa);
            }
        }
        if (p.rejected) p.rejected[idx] = rejected;
        if (DENSE) p.snap_count[idx] = next_j;
        active = false;
    };
    auto begin = [&](long long i) {
        idx = i;
        const long long n = p.n;
        t = 0.0;
        r = p.in[0 * n + i];
        th = p.in[1 * n + i];
        ph = p.in[2 * n + i];
        pr = p.in[3 * n + i];
        pth = p.in[4 * n + i];
        L = p.in[5 * n + i];
        bool y0_inside = true;
        if (METRIC == METRIC_TABG) {
            TabgFields F;
            y0_inside = tabg_fields_cold(p.tgm, r, th, F);
            const TabgAux A = tabg_aux(F.v, pr, pth, L, 0.0);                        // mass shell (5): A.W = beta^k p_k here
            E = fma(F.v[0], sqrt(p.kappa + A.gpp), -A.W);
        } else if (METRIC == METRIC_TAB) {
            TabFields F;
            y0_inside = tab_fields_cold(p.tm, r, th, F);
            E = fma(F.al, sqrt(p.kappa + pr * pr / F.g11 + pth * pth / F.g22 + L * L / F.g33), -F.be * L);   // mass shell (5)
        } else {
            E = energy_3p1(bh, r, th, pr, pth, L, p.kappa);
        }
        ct = cr = cth = cph = cpr = cpth = 0.0;
        h = p.h0;
        tau = 0.0;
        steps = attempts = rejected = 0;
        crossed = false;
        active = true;
        next_j = 0;
        if (!(r >= p.r_capture)) { E = kTab ? __longlong_as_double(0x7ff8000000000000LL) : E; finish(ST_CAPTURED); return; }   // B1
        if (kTab) {                                                              // T4 on y0: non-finite input, then the domain
            if (!all_finite6(r, th, ph, pr, pth, L)) { E = __longlong_as_double(0x7ff8000000000000LL); finish(ST_NUMERIC); return; }
            if (!y0_inside) { E = __longlong_as_double(0x7ff8000000000000LL); finish(ST_OUTSIDE); return; }
        }
        if (!all_finite6(r, th, ph, pr, pth, E)) { finish(ST_NUMERIC); return; }
        if (DENSE) { write_record(0, t, r, th, ph, pr, pth); next_j = 1; }      // record 0 = y0 (tau = 0)
        if (r > p.r_escape) { finish(ST_ESCAPED); return; }
        if (p.max_attempts == 0) { finish(ST_MAXSTEPS); return; }
        rhs_metric<METRIC>(p, r, th, pr, pth, E, L, k1);
    };

    for (;;) {
        // --- work queue (A5) ------------------------------------------------------------------
        unsigned idle = __ballot_sync(kFull, !active);
        if (idle) {
            if (!exhausted) {
                const int cnt = __popc(idle);
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(p.counter, (unsigned long long)cnt);
                base = __shfl_sync(kFull, base, 0);
                if (!active) {
                    const long long cand = (long long)base + __popc(idle & ((1u << lane) - 1u));
                    if (cand < p.n) begin(cand);
                }
                if ((long long)base + cnt >= p.n) exhausted = true;
                idle = __ballot_sync(kFull, !active);
            }
            if (idle == kFull) {
                if (exhausted) break;
                continue;
            }
        }

        // --- one attempt of size h (every lane; idle lanes compute on stale state) ----------------------
        const bool last = tau + 1.01 * h >= p.tau_end;                           // land on the final time
        if (last) h = p.tau_end - tau;
        Deriv d;
        double sr, sth, spr, spth;
        const K4 q1 = k4_of(k1);
        double s5t = dp::b1 * k1.t, s5p = dp::b1 * k1.ph;                        // b5 . k for the cyclic t, phi
        double set_ = dp::e1 * k1.t, sep = dp::e1 * k1.ph;                       // (b5 - b4) . k
        double sdt = 0, sdp = 0;                                                 // DENSE: d . k for t, phi
        if (DENSE) { sdt = dp::d1 * k1.t; sdp = dp::d1 * k1.ph; }
        // stage 2
        sr = fma(h * dp::a21, q1.r, r); sth = fma(h * dp::a21, q1.th, th);
        spr = fma(h * dp::a21, q1.pr, pr); spth = fma(h * dp::a21, q1.pth, pth);
        bool cap = false;
        int ev = 0;                      // tabulated metrics: first event in evaluation order (capture before domain exit, T7)
        auto evaluate = [&](Deriv& out) {
            const bool in = rhs_metric<METRIC>(p, sr, sth, spr, spth, E, L, out);
            if (kTab) {
                if (!ev) ev = !(sr >= p.r_capture) ? ST_CAPTURED : (!in ? ST_OUTSIDE : 0);
            } else {
                cap |= !(sr >= p.r_capture);
            }
        };
        evaluate(d);
        const K4 q2 = k4_of(d);
        // stage 3
        sr = fma(h, fma(dp::a32, q2.r, dp::a31 * q1.r), r); sth = fma(h, fma(dp::a32, q2.th, dp::a31 * q1.th), th);
        spr = fma(h, fma(dp::a32, q2.pr, dp::a31 * q1.pr), pr); spth = fma(h, fma(dp::a32, q2.pth, dp::a31 * q1.pth), pth);
        evaluate(d);
        const K4 q3 = k4_of(d);
        s5t = fma(dp::b3, d.t, s5t); s5p = fma(dp::b3, d.ph, s5p);
        if (DENSE) { sdt = fma(dp::d3, d.t, sdt); sdp = fma(dp::d3, d.ph, sdp); }
        set_ = fma(dp::e3, d.t, set_); sep = fma(dp::e3, d.ph, sep);
        // stage 4
#define GEO_S4(c) fma(dp::a43, q3.c, fma(dp::a42, q2.c, dp::a41 * q1.c))
        sr = fma(h, GEO_S4(r), r); sth = fma(h, GEO_S4(th), th); spr = fma(h, GEO_S4(pr), pr); spth = fma(h, GEO_S4(pth), pth);
#undef GEO_S4
        evaluate(d);
        const K4 q4 = k4_of(d);
        s5t = fma(dp::b4, d.t, s5t); s5p = fma(dp::b4, d.ph, s5p);
        if (DENSE) { sdt = fma(dp::d4, d.t, sdt); sdp = fma(dp::d4, d.ph, sdp); }
        set_ = fma(dp::e4, d.t, set_); sep = fma(dp::e4, d.ph, sep);
        // stage 5
#define GEO_S5(c) fma(dp::a54, q4.c, fma(dp::a53, q3.c, fma(dp::a52, q2.c, dp::a51 * q1.c)))
        sr = fma(h, GEO_S5(r), r); sth = fma(h, GEO_S5(th), th); spr = fma(h, GEO_S5(pr), pr); spth = fma(h, GEO_S5(pth), pth);
#undef GEO_S5
        evaluate(d);
        const K4 q5 = k4_of(d);
        s5t = fma(dp::b5, d.t, s5t); s5p = fma(dp::b5, d.ph, s5p);
        if (DENSE) { sdt = fma(dp::d5, d.t, sdt); sdp = fma(dp::d5, d.ph, sdp); }
        set_ = fma(dp::e5, d.t, set_); sep = fma(dp::e5, d.ph, sep);
        // stage 6
#define GEO_S6(c) fma(dp::a65, q5.c, fma(dp::a64, q4.c, fma(dp::a63, q3.c, fma(dp::a62, q2.c, dp::a61 * q1.c))))
        sr = fma(h, GEO_S6(r), r); sth = fma(h, GEO_S6(th), th); spr = fma(h, GEO_S6(pr), pr); spth = fma(h, GEO_S6(pth), pth);
#undef GEO_S6
        evaluate(d);
        const K4 q6 = k4_of(d);
        s5t = fma(dp::b6, d.t, s5t); s5p = fma(dp::b6, d.ph, s5p);
        if (DENSE) { sdt = fma(dp::d6, d.t, sdt); sdp = fma(dp::d6, d.ph, sdp); }
        set_ = fma(dp::e6, d.t, set_); sep = fma(dp::e6, d.ph, sep);
        // 5th-order solution, Kahan-compensated (committed only on acceptance); stage 7 sits on it
#define GEO_B5(c) fma(dp::b6, q6.c, fma(dp::b5, q5.c, fma(dp::b4, q4.c, fma(dp::b3, q3.c, dp::b1 * q1.c))))
        double nt, nr, nth, nph, npr, npth, dt, dr, dth, dph, dpr, dpth;
        kahan<false>(t, ct, h, s5t, nt, dt);
        kahan<false>(r, cr, h, GEO_B5(r), nr, dr);
        kahan<false>(th, cth, h, GEO_B5(th), nth, dth);
        kahan<false>(ph, cph, h, s5p, nph, dph);
        kahan<false>(pr, cpr, h, GEO_B5(pr), npr, dpr);
        kahan<false>(pth, cpth, h, GEO_B5(pth), npth, dpth);
#undef GEO_B5
        const bool fin6 = all_finite6(nt, nr, nth, nph, npr, npth);
        Deriv k7;
        const bool in7 = rhs_metric<METRIC>(p, nr, nth, npr, npth, E, L, k7);
        if (kTab) {                                                              // end point: capture, finiteness, then the domain
            if (!ev) ev = !(nr >= p.r_capture) ? ST_CAPTURED : ((fin6 && !in7) ? ST_OUTSIDE : 0);
            cap = ev != 0;
        } else {
            cap |= !(nr >= p.r_capture);                                         // B2: end point
        }
        // error estimate h (b5 - b4) . k, scaled per component; a NaN sticks in the max
#define GEO_E(c) fma(dp::e7, k7.c, fma(dp::e6, q6.c, fma(dp::e5, q5.c, fma(dp::e4, q4.c, fma(dp::e3, q3.c, dp::e1 * q1.c)))))
        double err = 0.0, ec;
        ec = scaled_err(h * fma(dp::e7, k7.t, set_), fma(p.rtol, fmax(fabs(t), fabs(nt)), p.atol));       if (!(ec <= err)) err = ec;
        ec = scaled_err(h * GEO_E(r), fma(p.rtol, fmax(fabs(r), fabs(nr)), p.atol));                        if (!(ec <= err)) err = ec;
        ec = scaled_err(h * GEO_E(th), fma(p.rtol, fmax(fabs(th), fabs(nth)), p.atol));                     if (!(ec <= err)) err = ec;
        ec = scaled_err(h * fma(dp::e7, k7.ph, sep), fma(p.rtol, fmax(fabs(ph), fabs(nph)), p.atol));      if (!(ec <= err)) err = ec;
        ec = scaled_err(h * GEO_E(pr), fma(p.rtol, fmax(fabs(pr), fabs(npr)), p.atol));                     if (!(ec <= err)) err = ec;
        ec = scaled_err(h * GEO_E(pth), fma(p.rtol, fmax(fabs(pth), fabs(npth)), p.atol));                  if (!(ec <= err)) err = ec;
#undef GEO_E
        double fac = err > 0.0 ? 0.9 * inv_fifth_root(err) : (err == 0.0 ? 5.0 : 0.2);   // NaN estimate: shrink
        if (!(fac >= 0.2)) fac = 0.2;
        if (fac > 5.0) fac = 5.0;
        if (p.fixed_step) { fac = 1.0; err = fin6 ? 0.0 : err; }

        if (active) {
            ++attempts;
            if (cap) {
                finish(kTab ? ev : ST_CAPTURED);                 // attempt not taken
            } else if (!fin6 || !(err <= 1.0)) {                                 // reject
                ++rejected;
                h *= fmin(fac, 1.0);
                // a non-finite attempt at a FIXED step can never succeed (same h, same NaN), and a step that has
                // shrunk to zero cannot advance: both end the particle like a step below h_min (reading A2)
                if ((p.fixed_step && !fin6) || !(fabs(h) >= p.h_min) || !(fabs(h) > 0.0)) finish(ST_NUMERIC);
                else if (attempts >= p.max_attempts) finish(ST_MAXSTEPS);
            } else {
                if (!crossed) {                                                  // B5
                    const double half_pi = 1.5707963267948966;
                    const double d0 = th - half_pi, d1 = nth - half_pi;
                    if (d0 * d1 < 0.0) {
                        crossed = true;
                        eqc = r + (nr - r) * (half_pi - th) / (nth - th);
                    }
                }
                const double tau_new = last ? p.tau_end : tau + h;               // the final time is landed on exactly
                if (DENSE) {                                                     // A3: every record time in (tau, tau_new]
                    double tj = (double)next_j * p.snap_dtau;
                    if (tj <= tau_new) {
                        // h sum_i d_i k_i per component (t, phi from the stage sums carried for them)
#define GEO_D(c) fma(dp::d7, k7.c, fma(dp::d6, q6.c, fma(dp::d5, q5.c, fma(dp::d4, q4.c, fma(dp::d3, q3.c, dp::d1 * q1.c)))))
                        const double hdt = h * fma(dp::d7, k7.t, sdt), hdp = h * fma(dp::d7, k7.ph, sdp);
                        const double hdr = h * GEO_D(r), hdth = h * GEO_D(th), hdpr = h * GEO_D(pr), hdpth = h * GEO_D(pth);
#undef GEO_D
                        const double ih = 1.0 / h;
                        do {
                            const double theta = (tj - tau) * ih;
                            write_record(next_j,
                                         contd5(theta, t, nt, h * k1.t, h * k7.t, hdt), contd5(theta, r, nr, h * q1.r, h * k7.r, hdr),
                                         contd5(theta, th, nth, h * q1.th, h * k7.th, hdth), contd5(theta, ph, nph, h * k1.ph, h * k7.ph, hdp),
                                         contd5(theta, pr, npr, h * q1.pr, h * k7.pr, hdpr), contd5(theta, pth, npth, h * q1.pth, h * k7.pth, hdpth));
                            ++next_j;
                            tj = (double)next_j * p.snap_dtau;
                        } while (tj <= tau_new);
                    }
                }
                t = nt; r = nr; th = nth; ph = nph; pr = npr; pth = npth;
                ct = dt; cr = dr; cth = dth; cph = dph; cpr = dpr; cpth = dpth;
                k1 = k7;                                                         // first same as last
                ++steps;
                tau = tau_new;
                h *= fac;
                if (r > p.r_escape) finish(ST_ESCAPED);                          // B3
                else if (last || attempts >= p.max_attempts) finish(ST_MAXSTEPS);   // final time / cap
            }
        }
    }
}

}  // namespace geo
