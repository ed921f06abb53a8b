// geo_ks_rk45.cuh -- the adaptive Dormand-Prince 5(4) stepper (readings A1-A3) in the Cartesian Kerr-Schild
// chart of geo_ks.cuh (SURVEY 8(f).3 second clause): DESIGN.md reading K6.  Same pair, controller, landing rule and
// continuous extension as geo_rk45.cuh (whose constants and helpers it uses); the seven evolving components
// (t~, x, y, z, p_x, p_y, p_z) enter the error norm.  Two rules are this chart's own:
//   K6a  step cap  h <- min(h, r / (4 |dx/dtau|)), dx/dtau = k_1 (not in fixed-step mode): far from the hole the geodesics
//        are straight lines here, the error estimate vanishes and the controller alone would let a step jump over the hole;
//   K6b  the capture test runs on y0 and on the END POINT of an attempt, not on the stage points: the chart is regular
//        through the horizon, and the stage points of a step along a tight orbit cut the chord (they dip below the orbit's
//        radius by r (dphi)^2 / 8), which would capture rays that skim the prograde photon orbit.
// With per-ray step control in this chart every pixel class of the configs[2] image equals the closed form: the polar-axis
// columns where the fixed-step Boyer-Lindquist path fails, and the prograde edge of the shadow where the fixed-step path of
// this chart fails.
#pragma once
#include "geo_ks.cuh"
#include "geo_rk45.cuh"

namespace geo {

struct KsAdaptiveParams {
    const double* in;   // [6][n]  x, y, z, p_x, p_y, p_z
    long long n;
    double h0, rtol, atol, h_min, tau_end;
    int fixed_step;
    int max_attempts;
    double r_capture, r_escape, kappa;
    double* fin;        // [8][n]
    int* status;
    long long* steps_done;
    double* eq_cross_r;
    double* health;
    int* rejected;
    unsigned long long* counter;
    double snap_dtau;
    double* snaps;
    long long snap_cap;
    unsigned snap_mask;
    int ncomp;
    int* snap_count;
    KsHole bh;
};

// the six components that feed back into the right-hand side
struct K6 {
    double x, y, z, px, py, pz;
};
__device__ __forceinline__ K6 k6_of(const KsDeriv& d) { return K6{d.x, d.y, d.z, d.px, d.py, d.pz}; }

#define GEO_KS_FOR6(M) M(x) M(y) M(z) M(px) M(py) M(pz)

template <bool DENSE>
__global__ void __launch_bounds__(kBlock, DENSE ? 2 : 3) geo_ks_rk45_kernel(const __grid_constant__ KsAdaptiveParams p) {
    const unsigned lane = threadIdx.x & 31u;
    const KsHole& bh = p.bh;
    long long idx = -1;
    bool active = false, exhausted = false;
    double t = 0, E = 0, ct = 0;
    K6 Y{0, 0, 0, 0, 0, 0}, Cc{0, 0, 0, 0, 0, 0};                   // state and its Kahan error terms (reading P1)
    double ry = 0;                                                   // r(x, y, z) of the current state
    double h = p.h0, tau = 0;
    KsDeriv k1;                                                      // f(y): first same as last
    k1.t = k1.x = k1.y = k1.z = k1.px = k1.py = k1.pz = 0;
    int steps = 0, attempts = 0, rejected = 0;
    double eqc = 0;
    bool crossed = false;
    int next_j = 0;

    auto write_record = [&](int j, double rt, const K6& s) {
        if (j < p.snap_cap) {
            double* dst = p.snaps + ((size_t)idx * (size_t)p.snap_cap + (size_t)j) * p.ncomp;
            store_record_global(dst, p.snap_mask, rt, s.x, s.y, s.z, E, s.px, s.py, s.pz);
        }
    };
    auto finish = [&](int st) {
        long long n = p.n;
        asm volatile("" : "+l"(n));
        p.fin[0 * n + idx] = t;
        p.fin[1 * n + idx] = Y.x;
        p.fin[2 * n + idx] = Y.y;
        p.fin[3 * n + idx] = Y.z;
        p.fin[4 * n + idx] = E;
        p.fin[5 * n + idx] = Y.px;
        p.fin[6 * n + idx] = Y.py;
        p.fin[7 * n + idx] = Y.pz;
        p.status[idx] = st;
        p.steps_done[idx] = (long long)steps;
        if (p.eq_cross_r) p.eq_cross_r[idx] = crossed ? eqc : __longlong_as_double(0x7ff8000000000000LL);
        if (p.health) p.health[idx] = health_ks(bh, Y.x, Y.y, Y.z, Y.px, Y.py, Y.pz, E, p.kappa);
        if (p.rejected) p.rejected[idx] = rejected;
        if (DENSE) p.snap_count[idx] = next_j;
        active = false;
    };
    auto begin = [&](long long i) {
        idx = i;
        const long long n = p.n;
        t = 0.0;
        Y.x = p.in[0 * n + i];
        Y.y = p.in[1 * n + i];
        Y.z = p.in[2 * n + i];
        Y.px = p.in[3 * n + i];
        Y.py = p.in[4 * n + i];
        Y.pz = p.in[5 * n + i];
        E = energy_ks(bh, Y.x, Y.y, Y.z, Y.px, Y.py, Y.pz, p.kappa);
        ct = 0.0;
        Cc = K6{0, 0, 0, 0, 0, 0};
        h = p.h0;
        tau = 0.0;
        steps = attempts = rejected = 0;
        crossed = false;
        active = true;
        next_j = 0;
        ry = radius_ks(bh, Y.x, Y.y, Y.z);
        if (!(ry >= p.r_capture)) { finish(ST_CAPTURED); return; }                                   // B1 / K2
        if (!all_finite6(Y.x, Y.y, Y.z, Y.px, Y.py, Y.pz) || !all_finite6(E, 0, 0, 0, 0, 0)) { finish(ST_NUMERIC); return; }
        if (DENSE) { write_record(0, t, Y); next_j = 1; }
        if (ry > p.r_escape) { finish(ST_ESCAPED); return; }
        if (p.max_attempts == 0) { finish(ST_MAXSTEPS); return; }
        double r0;
        rhs_ks(bh, Y.x, Y.y, Y.z, Y.px, Y.py, Y.pz, E, k1, r0);
    };

    for (;;) {
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
        if (!p.fixed_step) {                                                     // K6a
            const double v2 = fma(k1.x, k1.x, fma(k1.y, k1.y, k1.z * k1.z));
            const double hcap = (0.25 * ry) * rsqrt_c(v2);                       // (v2 = 0: +inf seed -> NaN, no cap)
            if (h > hcap) h = hcap;
        }
        const bool last = tau + 1.01 * h >= p.tau_end;
        if (last) h = p.tau_end - tau;
        KsDeriv d;
        K6 s;
        double rs;
        const K6 q1 = k6_of(k1);
        double s5t = dp::b1 * k1.t, set_ = dp::e1 * k1.t, sdt = 0;
        if (DENSE) sdt = dp::d1 * k1.t;
        // stage 2
#define GEO_ST(c) s.c = fma(h * dp::a21, q1.c, Y.c);
        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
        rhs_ks(bh, s.x, s.y, s.z, s.px, s.py, s.pz, E, d, rs);
        const K6 q2 = k6_of(d);
        // stage 3
#define GEO_ST(c) s.c = fma(h, fma(dp::a32, q2.c, dp::a31 * q1.c), Y.c);
        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
        rhs_ks(bh, s.x, s.y, s.z, s.px, s.py, s.pz, E, d, rs);
        const K6 q3 = k6_of(d);
        s5t = fma(dp::b3, d.t, s5t); set_ = fma(dp::e3, d.t, set_);
        if (DENSE) sdt = fma(dp::d3, d.t, sdt);
        // stage 4
#define GEO_ST(c) s.c = fma(h, fma(dp::a43, q3.c, fma(dp::a42, q2.c, dp::a41 * q1.c)), Y.c);
        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
        rhs_ks(bh, s.x, s.y, s.z, s.px, s.py, s.pz, E, d, rs);
        const K6 q4 = k6_of(d);
        s5t = fma(dp::b4, d.t, s5t); set_ = fma(dp::e4, d.t, set_);
        if (DENSE) sdt = fma(dp::d4, d.t, sdt);
        // stage 5
#define GEO_ST(c) s.c = fma(h, fma(dp::a54, q4.c, fma(dp::a53, q3.c, fma(dp::a52, q2.c, dp::a51 * q1.c))), Y.c);
        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
        rhs_ks(bh, s.x, s.y, s.z, s.px, s.py, s.pz, E, d, rs);
        const K6 q5 = k6_of(d);
        s5t = fma(dp::b5, d.t, s5t); set_ = fma(dp::e5, d.t, set_);
        if (DENSE) sdt = fma(dp::d5, d.t, sdt);
        // stage 6
#define GEO_ST(c) s.c = fma(h, fma(dp::a65, q5.c, fma(dp::a64, q4.c, fma(dp::a63, q3.c, fma(dp::a62, q2.c, dp::a61 * q1.c)))), Y.c);
        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
        rhs_ks(bh, s.x, s.y, s.z, s.px, s.py, s.pz, E, d, rs);
        const K6 q6 = k6_of(d);
        s5t = fma(dp::b6, d.t, s5t); set_ = fma(dp::e6, d.t, set_);
        if (DENSE) sdt = fma(dp::d6, d.t, sdt);
        // 5th-order solution, Kahan-compensated (committed only on acceptance); stage 7 sits on it
        double nt, dct;
        K6 N, Dc;
        kahan<false>(t, ct, h, s5t, nt, dct);
#define GEO_ST(c) kahan<false>(Y.c, Cc.c, h, fma(dp::b6, q6.c, fma(dp::b5, q5.c, fma(dp::b4, q4.c, fma(dp::b3, q3.c, dp::b1 * q1.c)))), N.c, Dc.c);
        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
        const bool fin7 = all_finite6(N.x, N.y, N.z, N.px, N.py, N.pz) && all_finite6(nt, 0, 0, 0, 0, 0);
        KsDeriv k7;
        double rn;
        rhs_ks(bh, N.x, N.y, N.z, N.px, N.py, N.pz, E, k7, rn);
        const bool cap = !(rn >= p.r_capture);                                   // K6b: end point only
        // error estimate h (b5 - b4) . k, scaled per component; a NaN sticks in the max
        double err = 0.0, ec;
        ec = scaled_err(h * fma(dp::e7, k7.t, set_), fma(p.rtol, fmax(fabs(t), fabs(nt)), p.atol));
        if (!(ec <= err)) err = ec;
#define GEO_ST(c)                                                                                                                        \
        ec = scaled_err(h * fma(dp::e7, k7.c, fma(dp::e6, q6.c, fma(dp::e5, q5.c, fma(dp::e4, q4.c, fma(dp::e3, q3.c, dp::e1 * q1.c))))), \
                        fma(p.rtol, fmax(fabs(Y.c), fabs(N.c)), p.atol));                                                                 \
        if (!(ec <= err)) err = ec;
        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
        double fac = err > 0.0 ? 0.9 * inv_fifth_root(err) : (err == 0.0 ? 5.0 : 0.2);
        if (!(fac >= 0.2)) fac = 0.2;
        if (fac > 5.0) fac = 5.0;
        if (p.fixed_step) { fac = 1.0; err = fin7 ? 0.0 : err; }

        if (active) {
            ++attempts;
            if (cap) {
                finish(ST_CAPTURED);                                             // attempt not taken
            } else if (!fin7 || !(err <= 1.0)) {                                 // reject
                ++rejected;
                h *= fmin(fac, 1.0);
                if ((p.fixed_step && !fin7) || !(fabs(h) >= p.h_min) || !(fabs(h) > 0.0)) finish(ST_NUMERIC);
                else if (attempts >= p.max_attempts) finish(ST_MAXSTEPS);
            } else {
                if (!crossed && Y.z * N.z < 0.0) {                               // K3
                    crossed = true;
                    eqc = ry + (rn - ry) * (0.0 - Y.z) / (N.z - Y.z);
                }
                const double tau_new = last ? p.tau_end : tau + h;
                if (DENSE) {
                    double tj = (double)next_j * p.snap_dtau;
                    if (tj <= tau_new) {
                        const double hdt = h * fma(dp::d7, k7.t, sdt);
                        K6 hd;
#define GEO_ST(c) hd.c = h * fma(dp::d7, k7.c, fma(dp::d6, q6.c, fma(dp::d5, q5.c, fma(dp::d4, q4.c, fma(dp::d3, q3.c, dp::d1 * q1.c)))));
                        GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
                        const double ih = 1.0 / h;
                        do {
                            const double theta = (tj - tau) * ih;
                            K6 rec;
#define GEO_ST(c) rec.c = contd5(theta, Y.c, N.c, h * q1.c, h * k7.c, hd.c);
                            GEO_KS_FOR6(GEO_ST)
#undef GEO_ST
                            write_record(next_j, contd5(theta, t, nt, h * k1.t, h * k7.t, hdt), rec);
                            ++next_j;
                            tj = (double)next_j * p.snap_dtau;
                        } while (tj <= tau_new);
                    }
                }
                t = nt; ct = dct;
                Y = N; Cc = Dc;
                ry = rn;
                k1 = k7;
                ++steps;
                tau = tau_new;
                h *= fac;
                if (ry > p.r_escape) finish(ST_ESCAPED);
                else if (last || attempts >= p.max_attempts) finish(ST_MAXSTEPS);
            }
        }
    }
}

#undef GEO_KS_FOR6

}  // namespace geo
