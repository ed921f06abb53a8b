// geo_ks.cuh -- SURVEY 8(f).3, second clause: an analytic metric in HORIZON-PENETRATING, AXIS-REGULAR coordinates on the
// fixed-step RK4 path ("further analytic metrics / horizon-penetrating, axis-regular coordinates"; the paper's motivation
// for the 3+1 form).  Kerr in Cartesian Kerr-Schild coordinates (t~, x, y, z), DESIGN.md
// readings K1-K5:
//     g_{mu nu} = eta_{mu nu} + f l_mu l_nu,   f = 2 M r^3/(r^4 + a^2 z^2) = 2 M r / D,   D = sqrt(w^2 + 4 a^2 z^2),
//     l_mu = (1, (r x + a y)/(r^2+a^2), (r y - a x)/(r^2+a^2), z/r),   r^2 = (w + D)/2,   w = x^2 + y^2 + z^2 - a^2,
// i.e. line element (1) with  alpha^2 = 1/(1+f),  beta^i = f l_i/(1+f),  gamma_ij = delta_ij + f l_i l_j.
// It is the paper's metric (6) in another chart (oracle/geo_ks_oracle.cpp header; tests/test_oracle_ks.py pulls it back).
// Nothing is singular on the polar axis or at r = r_+: no trigonometry, no 1/sin^2, no 1/Delta.
//
// Hamilton's equations (3),(4) of H = 1/2 [ -(p_t - beta^k p_k)^2/alpha^2 + gamma^{ij} p_i p_j ], p_t = -E:
// with lP = E + l_j p_j (so that alpha^-2 (E + beta.p) = E + f lP = dt~/dtau):
//     dx^i/dtau = p_i - f lP l_i,     dp_i/dtau = 1/2 (d_i f) lP^2 + f lP p_j d_i l_j,     dE/dtau = 0.
// The gradients are collected so that no l_i, d_i r, d_i f or d_i l_j is formed on its own:
//     u = x p_x + y p_y,  v = y p_x - x p_y,  N = r u + a v,  l.p = N/A + z p_z / r            (A = r^2 + a^2)
//     d_i r = x_i r/D (i = x, y),  z A/(r D) (i = z);     1/2 d_i f = M/D [ d_i r (1 - 4 r^2/D) + 2 (r/D) x_i ]
//     p_j d_i l_j = d_i r K + { (r p_x - a p_y)/A, (r p_y + a p_x)/A, p_z/r },   K = (u - 2 r N/A)/A - z p_z / r^2
//  => dp_x/dtau = x G1 + G2 (r p_x - a p_y),  dp_y/dtau = y G1 + G2 (r p_y + a p_x),  dp_z/dtau = z G3 + (f lP / r) p_z,
//     G1 = c5 lP^2 + f lP (r/D) K,  G2 = f lP / A,  G3 = fz lP^2 + f lP (A/(r D)) K.
// 81 FP64 instructions + 3 MUFU per evaluation (1/D and 1/r each from one MUFU.RSQ64H seed with a cubic correction, D = disc/D,
// r = r^2/r; one cubic-Newton reciprocal for 1/A).
// The oracle differentiates f and l_mu entry by entry with the quotient rule -- different algebra, no shared code.
#pragma once
#include "geo_kernel.cuh"

namespace geo {

struct KsHole {
    double M, a, a2, twoM, four_a2;
};

// 1/sqrt(x) for finite normal x > 0, faithfully rounded: MUFU.RSQ64H seed y0 (relative error ~2^-20), then ONE cubic
// correction  y0 (1 + e/2 + 3 e^2/8),  e = 1 - x y0^2  (|e| <~ 2^-19: the neglected 5 e^3/16 is < 2^-58).  Five FP64
// instructions; sqrt(x) = x rsqrt(x) costs one more (<= 1.5 ulp).  No special-case path (garbage in, garbage out).
__device__ __forceinline__ double rsqrt_c(double x) {
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    const double e = fma(-(x * y0), y0, 1.0);
    return fma(y0, e * fma(0.375, e, 0.5), y0);
}

struct KsDeriv {
    double t, x, y, z, px, py, pz;
};

// One evaluation of the right-hand side; also returns r at the evaluation point (the capture guard of the stage points).
__device__ __forceinline__ void rhs_ks(const KsHole& bh, double x, double y, double z, double px, double py, double pz,
                                       double E, KsDeriv& d, double& r_out) {
    const double R2 = fma(z, z, fma(y, y, x * x));
    const double w = R2 - bh.a2;
    const double disc = fma(w, w, (z * z) * bh.four_a2);
    const double iD = rsqrt_c(disc);
    const double D = disc * iD;
    const double r2 = 0.5 * (w + D);
    const double ir = rsqrt_c(r2);
    const double r = r2 * ir;
    r_out = r;
    const double A = r2 + bh.a2;
    const double iA = rcp_nr(A);
    const double c1 = r * iD;                                // d_x r / x
    const double f = bh.twoM * c1;                           // 2 M r / D
    // l.p without the l_i
    const double u = fma(x, px, y * py);
    const double v = fma(y, px, -(x * py));
    const double N = fma(r, u, bh.a * v);
    const double NiA = N * iA;
    const double zpz = z * pz;
    const double t1 = zpz * ir;
    const double lP = E + (NiA + t1);
    const double flP = f * lP;
    const double G2 = flP * iA;
    const double flPir = flP * ir;
    d.t = E + flP;                                           // alpha^-2 (E + beta.p)
    d.x = fma(-G2, fma(r, x, bh.a * y), px);                 // p_x - f lP l_x
    d.y = fma(-G2, fma(r, y, -(bh.a * x)), py);
    d.z = fma(-flPir, z, pz);
    // gradients, collected
    const double c6 = (A * ir) * iD;                         // d_z r / z
    const double c7 = bh.M * iD;
    const double r2iD = r2 * iD;
    const double c3 = fma(-4.0, r2iD, 1.0);
    const double c5 = (c7 * c1) * fma(-4.0, r2iD, 3.0);      // (1/2 d_x f) / x
    const double fz = c7 * fma(c3, c6, c1 + c1);             // (1/2 d_z f) / z
    const double K = fma(-t1, ir, iA * fma(-(r + r), NiA, u));
    const double lP2 = lP * lP;
    const double G1 = fma(flP * c1, K, c5 * lP2);
    const double G3 = fma(flP * c6, K, fz * lP2);
    d.px = fma(x, G1, G2 * fma(r, px, -(bh.a * py)));
    d.py = fma(y, G1, G2 * fma(r, py, bh.a * px));
    d.pz = fma(z, G3, flPir * pz);
}

// --- cold-path helpers (IEEE sqrt / division; once per particle or per rare event) ------------------------------------
__device__ __noinline__ double radius_ks(const KsHole& bh, double x, double y, double z) {
    const double w = x * x + y * y + z * z - bh.a2;
    return sqrt(0.5 * (w + sqrt(w * w + bh.four_a2 * z * z)));
}

// 3+1 pieces at a point: f and l.p
__device__ __forceinline__ void f_and_lp(const KsHole& bh, double x, double y, double z, double px, double py, double pz,
                                         double& f, double& lp) {
    const double r = radius_ks(bh, x, y, z);
    const double r2 = r * r;
    f = bh.twoM * r2 * r / (r2 * r2 + bh.a2 * z * z);
    lp = ((r * x + bh.a * y) * px + (r * y - bh.a * x) * py) / (r2 + bh.a2) + z * pz / r;
}

// E = alpha sqrt(kappa + gamma^{ij} p_i p_j) - beta^k p_k: the mass shell eq.(5) PAPER.md:69 in the variables of eq.(1)
__device__ __noinline__ double energy_ks(const KsHole& bh, double x, double y, double z, double px, double py, double pz,
                                         double kappa) {
    double f, lp;
    f_and_lp(bh, x, y, z, px, py, pz, f, lp);
    const double opf = 1.0 + f;
    const double gpp = px * px + py * py + pz * pz - f * lp * lp / opf;     // gamma^{ij} p_i p_j
    return sqrt((kappa + gpp) / opf) - f * lp / opf;
}

// |2H + kappa|, 2H = -(E + beta.p)^2/alpha^2 + gamma^{ij} p_i p_j
__device__ __noinline__ double health_ks(const KsHole& bh, double x, double y, double z, double px, double py, double pz,
                                         double E, double kappa) {
    double f, lp;
    f_and_lp(bh, x, y, z, px, py, pz, f, lp);
    const double opf = 1.0 + f;
    const double Ebp = E + f * lp / opf;
    const double twoH = -Ebp * Ebp * opf + (px * px + py * py + pz * pz - f * lp * lp / opf);
    return fabs(twoH + kappa);
}

struct KsParams {
    const double* in;   // [6][n]  x, y, z, p_x, p_y, p_z
    long long n;
    double h, h_half, h_sixth;
    int nsteps;
    double r_capture, r_escape, kappa;
    // end-point TRIGGERS from R^2 = x^2 + y^2 + z^2, which brackets r: r^2 <= R^2 <= r^2 + a^2 (the decision is taken behind
    // the rare branch with radius_ks):  possible capture <=> !(R^2 >= cap_R2), cap_R2 = r_capture^2 + a^2 (r < rc implies it);
    // possible escape <=> R^2 > esc_R2, esc_R2 = r_escape^2 (r > re implies it).  A NaN triggers the capture side.
    double cap_R2, esc_R2;
    int use_queue;
    int snap_every;
    long long snap_cap;
    unsigned snap_mask;
    int ncomp;
    double* fin;        // [8][n]  t~, x, y, z, E, p_x, p_y, p_z
    int* status;
    long long* steps_done;
    double* eq_cross_r;
    double* health;
    double* snaps;
    int* snap_count;
    unsigned long long* counter;
    KsHole bh;
};

struct Lane7 {
    double t, x, y, z, px, py, pz;
};
struct KsLaneState {
    Lane7 y, c;
};

__device__ __forceinline__ bool all_finite7(const Lane7& y) {
    const int m = 0x7fffffff;
    const int a = max(max(__double2hiint(y.t) & m, __double2hiint(y.x) & m), __double2hiint(y.y) & m);
    const int b = max(max(__double2hiint(y.z) & m, __double2hiint(y.px) & m), max(__double2hiint(y.py) & m, __double2hiint(y.pz) & m));
    return max(a, b) < 0x7ff00000;
}

// The persistent kernel: same skeleton as geo_rk4_kernel (lane-local state in registers, double-buffered over a 2x
// unrolled step loop, ONE rare-event branch per step, work queue with a warp-aggregated atomic, direct 256-bit record
// stores) around the Cartesian right-hand side.  12 warps per SM at <= 168 registers.
template <int SNAP, bool PLAIN>
__global__ void __launch_bounds__(kBlock, 3)
geo_ks_rk4_kernel(const __grid_constant__ KsParams p) {
    const unsigned lane = threadIdx.x & 31u;
    const KsHole& bh = p.bh;

    KsLaneState A, B;
    A.y = Lane7{0, 0, 0, 0, 0, 0, 0}; A.c = A.y; B = A;
    double E = 0;
    long long idx = -1;
    auto active = [&]() { return idx >= 0; };
    bool exhausted = !p.use_queue;
    int steps = 0, snap_ctr = 0, snaps = 0;
    bool crossed = false;
    double* my_snaps = nullptr;

    auto emit_snapshot = [&](const Lane7& y) {
        if (snaps < p.snap_cap)
            store_record_global(my_snaps + (size_t)snaps * p.ncomp, p.snap_mask, y.t, y.x, y.y, y.z, E, y.px, y.py, y.pz);
        ++snaps;
    };
    auto finish = [&](int st, const Lane7& y, int nsteps_done) {
        long long n = p.n;
        asm volatile("" : "+l"(n));
        p.fin[0 * n + idx] = y.t;
        p.fin[1 * n + idx] = y.x;
        p.fin[2 * n + idx] = y.y;
        p.fin[3 * n + idx] = y.z;
        p.fin[4 * n + idx] = E;
        p.fin[5 * n + idx] = y.px;
        p.fin[6 * n + idx] = y.py;
        p.fin[7 * n + idx] = y.pz;
        p.status[idx] = st;
        p.steps_done[idx] = (long long)nsteps_done;
        if (p.eq_cross_r && !crossed) p.eq_cross_r[idx] = __longlong_as_double(0x7ff8000000000000LL);
        if (p.health) p.health[idx] = health_ks(bh, y.x, y.y, y.z, y.px, y.py, y.pz, E, p.kappa);
        if (SNAP != SNAP_NONE) p.snap_count[idx] = snaps;
        idx = -1;
    };
    auto begin = [&](long long i) {
        idx = i;
        const long long n = p.n;
        Lane7& y = A.y;
        y.t = 0.0;
        y.x = p.in[0 * n + i];
        y.y = p.in[1 * n + i];
        y.z = p.in[2 * n + i];
        y.px = p.in[3 * n + i];
        y.py = p.in[4 * n + i];
        y.pz = p.in[5 * n + i];
        E = energy_ks(bh, y.x, y.y, y.z, y.px, y.py, y.pz, p.kappa);
        A.c = Lane7{0, 0, 0, 0, 0, 0, 0};
        steps = 0;
        snap_ctr = p.snap_every;
        snaps = 0;
        crossed = false;
        if (SNAP != SNAP_NONE) my_snaps = p.snaps + (size_t)i * (size_t)p.snap_cap * p.ncomp;
        const double r0 = radius_ks(bh, y.x, y.y, y.z);
        if (!(r0 >= p.r_capture)) { finish(ST_CAPTURED, y, 0); return; }                      // B1 with r(x, y, z) (K2)
        if (!all_finite7(y) || !all_finite6(E, 0, 0, 0, 0, 0)) { finish(ST_NUMERIC, y, 0); return; }
        if (SNAP != SNAP_NONE) emit_snapshot(y);
        if (r0 > p.r_escape) { finish(ST_ESCAPED, y, 0); return; }
        if (p.nsteps == 0) { finish(ST_MAXSTEPS, y, 0); return; }
    };

    auto step = [&](const KsLaneState& cur, KsLaneState& nxt) {
        const double x = cur.y.x, y = cur.y.y, z = cur.y.z, px = cur.y.px, py = cur.y.py, pz = cur.y.pz;
        KsDeriv k;
        double rs;
        double at, ax, ay, az, apx, apy, apz;
        double sx, sy, sz, spx, spy, spz;
        rhs_ks(bh, x, y, z, px, py, pz, E, k, rs);
        at = k.t; ax = k.x; ay = k.y; az = k.z; apx = k.px; apy = k.py; apz = k.pz;
        sx = fma(p.h_half, k.x, x); sy = fma(p.h_half, k.y, y); sz = fma(p.h_half, k.z, z);
        spx = fma(p.h_half, k.px, px); spy = fma(p.h_half, k.py, py); spz = fma(p.h_half, k.pz, pz);

        rhs_ks(bh, sx, sy, sz, spx, spy, spz, E, k, rs);
        bool cap = !(rs >= p.r_capture);                                   // B2: stage point 2
        at = fma(2.0, k.t, at); ax = fma(2.0, k.x, ax); ay = fma(2.0, k.y, ay); az = fma(2.0, k.z, az);
        apx = fma(2.0, k.px, apx); apy = fma(2.0, k.py, apy); apz = fma(2.0, k.pz, apz);
        sx = fma(p.h_half, k.x, x); sy = fma(p.h_half, k.y, y); sz = fma(p.h_half, k.z, z);
        spx = fma(p.h_half, k.px, px); spy = fma(p.h_half, k.py, py); spz = fma(p.h_half, k.pz, pz);

        rhs_ks(bh, sx, sy, sz, spx, spy, spz, E, k, rs);
        cap |= !(rs >= p.r_capture);                                       // stage point 3
        at = fma(2.0, k.t, at); ax = fma(2.0, k.x, ax); ay = fma(2.0, k.y, ay); az = fma(2.0, k.z, az);
        apx = fma(2.0, k.px, apx); apy = fma(2.0, k.py, apy); apz = fma(2.0, k.pz, apz);
        sx = fma(p.h, k.x, x); sy = fma(p.h, k.y, y); sz = fma(p.h, k.z, z);
        spx = fma(p.h, k.px, px); spy = fma(p.h, k.py, py); spz = fma(p.h, k.pz, pz);

        rhs_ks(bh, sx, sy, sz, spx, spy, spz, E, k, rs);
        cap |= !(rs >= p.r_capture);                                       // stage point 4
        at += k.t; ax += k.x; ay += k.y; az += k.z; apx += k.px; apy += k.py; apz += k.pz;

        kahan<PLAIN>(cur.y.t, cur.c.t, p.h_sixth, at, nxt.y.t, nxt.c.t);
        kahan<PLAIN>(x, cur.c.x, p.h_sixth, ax, nxt.y.x, nxt.c.x);
        kahan<PLAIN>(y, cur.c.y, p.h_sixth, ay, nxt.y.y, nxt.c.y);
        kahan<PLAIN>(z, cur.c.z, p.h_sixth, az, nxt.y.z, nxt.c.z);
        kahan<PLAIN>(px, cur.c.px, p.h_sixth, apx, nxt.y.px, nxt.c.px);
        kahan<PLAIN>(py, cur.c.py, p.h_sixth, apy, nxt.y.py, nxt.c.py);
        kahan<PLAIN>(pz, cur.c.pz, p.h_sixth, apz, nxt.y.pz, nxt.c.pz);
        // end point: capture / escape triggers from R^2 (no square root in the accepted step)
        const double Rn2 = fma(nxt.y.z, nxt.y.z, fma(nxt.y.y, nxt.y.y, nxt.y.x * nxt.y.x));
        const bool cap_end = !(Rn2 >= p.cap_R2);
        const bool esc_end = Rn2 > p.esc_R2;
        const bool fin7 = all_finite7(nxt.y);
        const bool maybe_crossing = (__double2hiint(z) ^ __double2hiint(nxt.y.z)) < 0;     // K3 candidate: sign bits differ
        const int ns = steps + 1;
        bool rare = cap | cap_end | esc_end | !fin7 | maybe_crossing | (ns >= p.nsteps);
        if (SNAP != SNAP_NONE) rare |= (--snap_ctr == 0);
        steps = ns;

        if (__builtin_expect(rare && active(), 0)) {
            const double rn = radius_ks(bh, nxt.y.x, nxt.y.y, nxt.y.z);
            if (cap || !(rn >= p.r_capture)) {
                finish(ST_CAPTURED, cur.y, ns - 1);
            } else if (!fin7) {
                finish(ST_NUMERIC, cur.y, ns - 1);
            } else {
                if (!crossed && z * nxt.y.z < 0.0) {                       // K3: first sign change of z
                    crossed = true;
                    if (p.eq_cross_r) {
                        const double r0 = radius_ks(bh, x, y, z);
                        p.eq_cross_r[idx] = r0 + (rn - r0) * (0.0 - z) / (nxt.y.z - z);
                    }
                }
                if (SNAP != SNAP_NONE) {
                    if (snap_ctr == 0) { snap_ctr = p.snap_every; emit_snapshot(nxt.y); }
                }
                if (rn > p.r_escape) finish(ST_ESCAPED, nxt.y, ns);
                else if (ns >= p.nsteps) finish(ST_MAXSTEPS, nxt.y, ns);
            }
        }
    };

    if (!p.use_queue) {
        const long long i = (long long)blockIdx.x * kBlock + threadIdx.x;
        if (i < p.n) begin(i);
    }

    for (;;) {
        unsigned idle = __ballot_sync(kFull, !active());
        if (idle) {
            if (!exhausted) {
                const int cnt = __popc(idle);
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(p.counter, (unsigned long long)cnt);
                base = __shfl_sync(kFull, base, 0);
                if (!active()) {
                    const long long cand = (long long)base + __popc(idle & ((1u << lane) - 1u));
                    if (cand < p.n) begin(cand);
                }
                if ((long long)base + cnt >= p.n) exhausted = true;
                idle = __ballot_sync(kFull, !active());
            }
            if (idle == kFull) {
                if (exhausted) break;
                continue;
            }
        }
        step(A, B);
        step(B, A);
    }
}

}  // namespace geo
