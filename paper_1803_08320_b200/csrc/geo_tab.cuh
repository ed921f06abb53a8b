// geo_tab.cuh -- SURVEY 8(f).3: fixed-step RK4 geodesics through a NUMERICALLY GIVEN (tabulated) stationary,
// axisymmetric 3+1 metric -- the "numerical metrics" the paper gives as the reason for its 3+1 formulation
// (PAPER.md:31-33, 497).  One persistent kernel with the work queue, stop rules and Kahan update of the
// analytic-metric kernel (geo_kernel.cuh); what changes is the RHS evaluator: the five functions of eq.(8)
// -- lapse alpha, shift beta^phi, gamma_11, gamma_22, gamma_33 -- come from a table on a
// uniform (x^1, x^2) grid through the tensor-product cubic-convolution interpolant (Keys 1981, a = -1/2:
// C^1, exact on quadratics), and the derivatives in Hamilton's equations (3),(4) are the
// exact derivatives of that interpolant (readings T1-T5), so E and L are constants of motion.
//
//   H = 1/2 [ -(E + beta^phi L)^2/alpha^2 + p_1^2/gamma_11 + p_2^2/gamma_22 + L^2/gamma_33 ],  u^t = (E + beta^phi L)/alpha^2
//   dx^k/dtau = p_k/gamma_kk,  dphi/dtau = L/gamma_33 - beta^phi u^t,  dt/dtau = u^t
//   dp_k/dtau = u^t L d_k beta^phi - alpha (u^t)^2 d_k alpha + 1/2 sum_m d_k gamma_mm (p_m/gamma_mm)^2
//
// Table layout in HBM/L2 (built once by tab_pack_kernel from the caller's [5][n2][n1] array): node-major,
//   A[j][i] = (alpha, beta^phi, gamma_11, gamma_22) as one 32-byte record -> one 256-bit load per node,
//   B[j][i] = gamma_33                                                    -> four consecutive doubles per stencil row.
// One RHS evaluation reads the 4 x 4 stencil = 16 records of A + 16 doubles of B = 640 B per lane, ~23 32-B
// sectors; a whole table of 2053 x 517 nodes is 42 MB and lives in the 126 MB L2.  Per lane and evaluation:
// ~330 FP64 instructions (separable evaluation: 8 FMA per field and stencil row for the value and the
// x^1-derivative along x^1, then 3 FMA per row along x^2).  The stencil is read from the table (16 LDG.256 + 16
// LDG.64) only when the particle enters a new cell: between refills it sits in a per-lane on-chip cache (below).
// GEO_FLAG_TAB_GATHER selects the variant that gathers it on every evaluation (L1-wavefront-bound, 2.6x slower).
#pragma once
#include "geo_kernel.cuh"

namespace geo {

enum { ST_OUTSIDE = 4 };

struct TabMetric {
    const double4* A;   // [n2][n1] (alpha, beta^phi, gamma_11, gamma_22)
    const double* B;    // [n2][n1] gamma_33
    int n1, n2;
    double x1_0, d1, inv_d1, x2_0, d2, inv_d2;
};

struct TabParams {
    const double* in;   // [6][n] (x1, x2, phi, p_1, p_2, p_phi)
    long long n;
    double h, h_half, h_sixth;
    int nsteps;
    double r_capture, r_escape, kappa;
    double* fin;        // [8][n]
    int* status;
    long long* steps_done;
    double* eq_cross_r;
    double* health;
    unsigned long long* counter;
    // trajectory records (readings S1-S3): components (t, x1, x2, phi, E, p1, p2, L) by mask, particle-major
    int snap_every;
    long long snap_cap;
    unsigned snap_mask;
    int ncomp;
    double* snaps;
    int* snap_count;
    TabMetric m;
};

struct TabFields {
    double al, be, g11, g22, g33;          // values
    double al1, be1, g111, g221, g331;     // d/dx^1
    double al2, be2, g112, g222, g332;     // d/dx^2
};

__device__ __forceinline__ double4 ldg256(const double4* p) {
    double4 v;
    asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}

// cell index and in-cell coordinate along one direction (reading T2, T4): u = (x - x0)/d, i = floor(u), s = u - i.
// The quotient is formed with the reciprocal; when s falls within 2^-30 of a cell face it is redone with a true
// division, so the floor -- which decides the cell and the domain test -- is the oracle's.
__device__ __forceinline__ bool tab_cell(double x, double x0, double d, double inv_d, int n, int& i, double& s) {
    double u = (x - x0) * inv_d;
    int k = __double2int_rd(u);                // NaN -> 0: fails the domain test below
    double sf = u - (double)k;
    if (sf < 9.3e-10 || sf > 1.0 - 9.3e-10) {
        u = (x - x0) / d;
        k = __double2int_rd(u);
        sf = u - (double)k;
    }
    const bool inside = (k >= 1) & (k <= n - 3) & (u < 2.0e9) & (u > -2.0e9);
    i = min(max(k, 1), n - 3);                 // loads stay in bounds whatever the lane holds
    s = inside ? sf : 0.0;
    return inside;
}

// Keys weights of nodes i-1 .. i+2 and their derivatives with respect to x (= inv_d * d/ds)
__device__ __forceinline__ void keys_weights(double s, double inv_d, double w[4], double dw[4]) {
    const double s2 = s * s;
    w[0] = 0.5 * s * fma(s, 2.0 - s, -1.0);
    w[1] = fma(s2, fma(1.5, s, -2.5), 1.0);
    w[2] = 0.5 * s * fma(s, fma(-3.0, s, 4.0), 1.0);
    w[3] = 0.5 * s2 * (s - 1.0);
    const double hd = 0.5 * inv_d;
    dw[0] = hd * fma(s, fma(-3.0, s, 4.0), -1.0);
    dw[1] = hd * s * fma(9.0, s, -10.0);
    dw[2] = hd * fma(s, fma(-9.0, s, 8.0), 1.0);
    dw[3] = hd * s * fma(3.0, s, -2.0);
}

// Interpolated fields and their gradients at (x1, x2).  Returns false outside the domain (the values are then
// those of the nearest interior cell's stencil at s = 0 -- finite garbage that the caller discards).
__device__ __forceinline__ bool tab_fields(const TabMetric& m, double x1, double x2, TabFields& F) {
    int i, j;
    double s1, s2;
    const bool in1 = tab_cell(x1, m.x1_0, m.d1, m.inv_d1, m.n1, i, s1);
    const bool in2 = tab_cell(x2, m.x2_0, m.d2, m.inv_d2, m.n2, j, s2);
    double w1[4], dw1[4], w2[4], dw2[4];
    keys_weights(s1, m.inv_d1, w1, dw1);
    keys_weights(s2, m.inv_d2, w2, dw2);
    const long long base = (long long)(j - 1) * m.n1 + (i - 1);
    double v[5] = {0, 0, 0, 0, 0}, g1[5] = {0, 0, 0, 0, 0}, g2[5] = {0, 0, 0, 0, 0};
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const double4* ra = m.A + base + (long long)b * m.n1;
        const double* rb = m.B + base + (long long)b * m.n1;
        const double4 a0 = ldg256(ra), a1 = ldg256(ra + 1), a2 = ldg256(ra + 2), a3 = ldg256(ra + 3);
        const double b0 = __ldg(rb), b1 = __ldg(rb + 1), b2 = __ldg(rb + 2), b3 = __ldg(rb + 3);
        double rv[5], rd[5];      // value and x^1-derivative along this stencil row
#define GEO_ROW(k, c0, c1, c2, c3)                                                   \
        rv[k] = fma(w1[3], c3, fma(w1[2], c2, fma(w1[1], c1, w1[0] * c0)));          \
        rd[k] = fma(dw1[3], c3, fma(dw1[2], c2, fma(dw1[1], c1, dw1[0] * c0)));
        GEO_ROW(0, a0.x, a1.x, a2.x, a3.x)
        GEO_ROW(1, a0.y, a1.y, a2.y, a3.y)
        GEO_ROW(2, a0.z, a1.z, a2.z, a3.z)
        GEO_ROW(3, a0.w, a1.w, a2.w, a3.w)
        GEO_ROW(4, b0, b1, b2, b3)
#undef GEO_ROW
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            v[k] = fma(w2[b], rv[k], v[k]);
            g1[k] = fma(w2[b], rd[k], g1[k]);
            g2[k] = fma(dw2[b], rv[k], g2[k]);
        }
    }
    F.al = v[0]; F.be = v[1]; F.g11 = v[2]; F.g22 = v[3]; F.g33 = v[4];
    F.al1 = g1[0]; F.be1 = g1[1]; F.g111 = g1[2]; F.g221 = g1[3]; F.g331 = g1[4];
    F.al2 = g2[0]; F.be2 = g2[1]; F.g112 = g2[2]; F.g222 = g2[3]; F.g332 = g2[4];
    return in1 & in2;
}

// ---- per-lane stencil cache ------------------------------------------------------------------------------------
// A particle stays in one grid cell for many evaluations (a step moves it by h |dx/dtau| << d), so the 4 x 4 x 5
// stencil of its current cell is kept on chip and refilled from the table only when the cell index changes: the
// stencils of the first R fields in REGISTERS (statically indexed after unrolling; the refill writes them under the
// lane's predicate), those of the other S = 5 - R fields in shared memory, column-major [16 S][kTabBlock] doubles per
// CTA (lane l owns column l: its 64-bit accesses are conflict-free, 2 wavefronts per warp instruction instead of
// the 32 of a gather).  Element (b, a, f) of the shared part sits at row (b*4 + a) S + (f - R).
// Measured (profiles/r01_tab4.md): R = 0 7.20e9, R = 1 7.38e9, R = 2 7.26e9, R = 3 6.25e9 (spills), R = 5 6.85e9 steps/s.
#ifndef GEO_TAB_BLOCK
#define GEO_TAB_BLOCK 128
#endif
#ifndef GEO_TAB_CTAS
#define GEO_TAB_CTAS 2
#endif
#ifndef GEO_TAB_REGFIELDS
#define GEO_TAB_REGFIELDS 1
#endif
constexpr int kTabBlock = GEO_TAB_BLOCK;      // threads per CTA of the tabulated-metric kernels
constexpr int kTabRegFields = GEO_TAB_REGFIELDS;
constexpr int kTabSmemRows = 16 * (5 - kTabRegFields);

template <int R>
__device__ __forceinline__ bool tab_fields_hybrid(const TabMetric& m, double x1, double x2, TabFields& F, int& ci, int& cj,
                                                  double* col, double (&rs)[16][R > 0 ? R : 1]) {
    constexpr int S = 5 - R;
    int i, j;
    double s1, s2;
    const bool in1 = tab_cell(x1, m.x1_0, m.d1, m.inv_d1, m.n1, i, s1);
    const bool in2 = tab_cell(x2, m.x2_0, m.d2, m.inv_d2, m.n2, j, s2);
    if (i != ci || j != cj) {
        const long long base = (long long)(j - 1) * m.n1 + (i - 1);
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double4* ra = m.A + base + (long long)b * m.n1;
            const double* rb = m.B + base + (long long)b * m.n1;
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const double4 v = ldg256(ra + a);
                const double vals[5] = {v.x, v.y, v.z, v.w, __ldg(rb + a)};
#pragma unroll
                for (int f = 0; f < 5; ++f) {
                    if (f < R) rs[b * 4 + a][f < R ? f : 0] = vals[f];
                    else col[((b * 4 + a) * S + (f - R)) * kTabBlock] = vals[f];
                }
            }
        }
        ci = i;
        cj = j;
    }
    double w1[4], dw1[4], w2[4], dw2[4];
    keys_weights(s1, m.inv_d1, w1, dw1);
    keys_weights(s2, m.inv_d2, w2, dw2);
    double v[5] = {0, 0, 0, 0, 0}, g1[5] = {0, 0, 0, 0, 0}, g2[5] = {0, 0, 0, 0, 0};
#pragma unroll
    for (int b = 0; b < 4; ++b) {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            double c[4];
#pragma unroll
            for (int a = 0; a < 4; ++a)
                c[a] = k < R ? rs[b * 4 + a][k < R ? k : 0] : col[((b * 4 + a) * S + (k - R)) * kTabBlock];
            const double rv = fma(w1[3], c[3], fma(w1[2], c[2], fma(w1[1], c[1], w1[0] * c[0])));
            const double rd = fma(dw1[3], c[3], fma(dw1[2], c[2], fma(dw1[1], c[1], dw1[0] * c[0])));
            v[k] = fma(w2[b], rv, v[k]);
            g1[k] = fma(w2[b], rd, g1[k]);
            g2[k] = fma(dw2[b], rv, g2[k]);
        }
    }
    F.al = v[0]; F.be = v[1]; F.g11 = v[2]; F.g22 = v[3]; F.g33 = v[4];
    F.al1 = g1[0]; F.be1 = g1[1]; F.g111 = g1[2]; F.g221 = g1[3]; F.g331 = g1[4];
    F.al2 = g2[0]; F.be2 = g2[1]; F.g112 = g2[2]; F.g222 = g2[3]; F.g332 = g2[4];
    return in1 & in2;
}

struct TabDeriv {
    double t, x1, x2, ph, p1, p2;
};

// Hamilton's equations of the 3+1 Hamiltonian in the interpolated fields (reading T3)
__device__ __forceinline__ void tab_rhs(const TabFields& F, double p1, double p2, double E, double L, TabDeriv& d) {
    const double W = fma(F.be, L, E);
    const double ut = W * rcp_nr(F.al * F.al);
    const double v1 = p1 * rcp_nr(F.g11), v2 = p2 * rcp_nr(F.g22), v3 = L * rcp_nr(F.g33);
    const double utL = ut * L, q = -F.al * ut * ut;
    const double h11 = 0.5 * v1 * v1, h22 = 0.5 * v2 * v2, h33 = 0.5 * v3 * v3;
    d.t = ut;
    d.x1 = v1;
    d.x2 = v2;
    d.ph = fma(-F.be, ut, v3);
    d.p1 = fma(utL, F.be1, fma(q, F.al1, fma(F.g111, h11, fma(F.g221, h22, F.g331 * h33))));
    d.p2 = fma(utL, F.be2, fma(q, F.al2, fma(F.g112, h11, fma(F.g222, h22, F.g332 * h33))));
}

__device__ __noinline__ bool tab_fields_cold(const TabMetric& m, double x1, double x2, TabFields& F) {
    return tab_fields(m, x1, x2, F);
}

// CACHE: per-lane stencil cache (kTabSmemRows * kTabBlock doubles = 64 KB of shared memory per CTA, 2 CTAs/SM);
// !CACHE: every evaluation gathers its stencil through L1/L2 (GEO_FLAG_TAB_GATHER, for comparison).
// SNAP: trajectory records (a separate instantiation: the stepping kernel has no register to spare).
template <bool PLAIN, bool CACHE, bool SNAP>
__global__ void __launch_bounds__(kTabBlock, CACHE ? GEO_TAB_CTAS : 3) geo_tab_rk4_kernel(const __grid_constant__ TabParams p) {
    extern __shared__ __align__(16) double stencil_smem[];
    double* const col = stencil_smem + threadIdx.x;
    int ci = -1, cj = -1;                                          // cell whose stencil the column holds
    const unsigned lane = threadIdx.x & 31u;
    const TabMetric& m = p.m;
    double rs[16][kTabRegFields > 0 ? kTabRegFields : 1];          // register-resident part of the stencil cache
    auto fields = [&](double a, double b, TabFields& F) -> bool {
        if (CACHE) return tab_fields_hybrid<kTabRegFields>(m, a, b, F, ci, cj, col, rs);
        return tab_fields(m, a, b, F);
    };
    long long idx = -1;
    bool active = false, exhausted = false;
    double t = 0, x1 = 0, x2 = 0, ph = 0, p1 = 0, p2 = 0, E = 0, L = 0;
    double ct = 0, c1 = 0, c2 = 0, cph = 0, cp1 = 0, cp2 = 0;     // Kahan error terms (reading P1)
    TabDeriv k1;                                                   // f(y), carried from the end-point evaluation
    k1.t = k1.x1 = k1.x2 = k1.ph = k1.p1 = k1.p2 = 0;
    int steps = 0;
    double eqc = 0;
    bool crossed = false;
    int snaps = 0, snap_ctr = 0;

    auto emit_record = [&]() {                                     // S1-S3: straight from registers, 256-bit stores
        if (snaps < p.snap_cap)
            store_record_global(p.snaps + ((size_t)idx * (size_t)p.snap_cap + (size_t)snaps) * p.ncomp, p.snap_mask,
                                t, x1, x2, ph, E, p1, p2, L);
        ++snaps;
    };
    auto finish = [&](int st) {
        long long n = p.n;
        asm volatile("" : "+l"(n));
        if (SNAP) p.snap_count[idx] = snaps;
        p.fin[0 * n + idx] = t;
        p.fin[1 * n + idx] = x1;
        p.fin[2 * n + idx] = x2;
        p.fin[3 * n + idx] = ph;
        p.fin[4 * n + idx] = E;
        p.fin[5 * n + idx] = p1;
        p.fin[6 * n + idx] = p2;
        p.fin[7 * n + idx] = L;
        p.status[idx] = st;
        p.steps_done[idx] = (long long)steps;
        const double qnan = __longlong_as_double(0x7ff8000000000000LL);
        if (p.eq_cross_r) p.eq_cross_r[idx] = crossed ? eqc : qnan;
        if (p.health) {
            TabFields F;
            double hv = qnan;
            if (tab_fields_cold(m, x1, x2, F) && (__double2hiint(E) & 0x7ff00000) != 0x7ff00000) {
                const double W = fma(F.be, L, E);
                hv = fabs(-(W * W) / (F.al * F.al) + p1 * p1 / F.g11 + p2 * p2 / F.g22 + L * L / F.g33 + p.kappa);
            }
            p.health[idx] = hv;
        }
        active = false;
    };
    auto begin = [&](long long i) {
        idx = i;
        const long long n = p.n;
        t = 0.0;
        x1 = p.in[0 * n + i];
        x2 = p.in[1 * n + i];
        ph = p.in[2 * n + i];
        p1 = p.in[3 * n + i];
        p2 = p.in[4 * n + i];
        L = p.in[5 * n + i];
        E = __longlong_as_double(0x7ff8000000000000LL);
        ct = c1 = c2 = cph = cp1 = cp2 = 0.0;
        steps = 0;
        crossed = false;
        active = true;
        snaps = 0;
        snap_ctr = p.snap_every;
        if (!(x1 >= p.r_capture)) { finish(ST_CAPTURED); return; }               // B1
        if (!all_finite6(x1, x2, ph, p1, p2, L)) { finish(ST_NUMERIC); return; }
        TabFields F;
        if (!tab_fields_cold(m, x1, x2, F)) { finish(ST_OUTSIDE); return; }      // T4 on y0
        E = fma(F.al, sqrt(p.kappa + p1 * p1 / F.g11 + p2 * p2 / F.g22 + L * L / F.g33), -F.be * L);   // mass shell (5)
        if ((__double2hiint(E) & 0x7ff00000) == 0x7ff00000) { finish(ST_NUMERIC); return; }
        if (SNAP) emit_record();                                                 // S1: slot 0 = y0
        if (x1 > p.r_escape) { finish(ST_ESCAPED); return; }
        if (p.nsteps == 0) { finish(ST_MAXSTEPS); return; }
        tab_rhs(F, p1, p2, E, L, k1);
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

        // --- one RK4 step (every lane; idle lanes compute on stale state, loads are clamped in bounds) ----
        // ev: first event in the oracle's order -- per evaluation point capture (B2) before domain exit (T4)
        // The four evaluations (stage points 2-4, end point) run through ONE copy of the evaluator (loop not
        // unrolled): unrolled, the step is ~9000 instructions and the warps stall on instruction fetch
        // (ncu: stall_no_instruction 1.8 per issue).
        int ev = 0;
        TabDeriv d = k1;
        double at = k1.t, a1 = k1.x1, a2 = k1.x2, aph = k1.ph, ap1 = k1.p1, ap2 = k1.p2;
        double nt = t, n1 = x1, n2 = x2, nph = ph, np1 = p1, np2 = p2, dt = ct, d1 = c1, d2 = c2, dph = cph, dp1 = cp1, dp2 = cp2;
#pragma unroll 1
        for (int s = 0; s < 4; ++s) {
            double e1, e2, ep1, ep2;                                   // evaluation point
            bool fin6 = true;
            if (s < 3) {
                const double c = s == 2 ? p.h : p.h_half;
                e1 = fma(c, d.x1, x1); e2 = fma(c, d.x2, x2);
                ep1 = fma(c, d.p1, p1); ep2 = fma(c, d.p2, p2);
            } else {
                // update (Kahan, reading P1); the end point's derivative is the next step's k1
                kahan<PLAIN>(t, ct, p.h_sixth, at, nt, dt);
                kahan<PLAIN>(x1, c1, p.h_sixth, a1, n1, d1);
                kahan<PLAIN>(x2, c2, p.h_sixth, a2, n2, d2);
                kahan<PLAIN>(ph, cph, p.h_sixth, aph, nph, dph);
                kahan<PLAIN>(p1, cp1, p.h_sixth, ap1, np1, dp1);
                kahan<PLAIN>(p2, cp2, p.h_sixth, ap2, np2, dp2);
                e1 = n1; e2 = n2; ep1 = np1; ep2 = np2;
                fin6 = all_finite6(nt, n1, n2, nph, np1, np2);
            }
            TabFields F;
            const bool in = fields(e1, e2, F);
            if (!ev) ev = !(e1 >= p.r_capture) ? ST_CAPTURED : (!fin6 ? ST_NUMERIC : (!in ? ST_OUTSIDE : 0));
            tab_rhs(F, ep1, ep2, E, L, d);
            if (s < 3) {
                const double w = s == 2 ? 1.0 : 2.0;                   // k1 + 2 k2 + 2 k3 + k4
                at = fma(w, d.t, at); a1 = fma(w, d.x1, a1); a2 = fma(w, d.x2, a2);
                aph = fma(w, d.ph, aph); ap1 = fma(w, d.p1, ap1); ap2 = fma(w, d.p2, ap2);
            }
        }

        if (active) {
            if (ev) {
                finish(ev);                                                      // step not taken
            } else {
                if (!crossed) {                                                  // B5
                    const double half_pi = 1.5707963267948966;
                    const double e0 = x2 - half_pi, e1 = n2 - half_pi;
                    if (e0 * e1 < 0.0) {
                        crossed = true;
                        eqc = x1 + (n1 - x1) * (half_pi - x2) / (n2 - x2);
                    }
                }
                t = nt; x1 = n1; x2 = n2; ph = nph; p1 = np1; p2 = np2;
                ct = dt; c1 = d1; c2 = d2; cph = dph; cp1 = dp1; cp2 = dp2;
                k1 = d;
                ++steps;
                if (SNAP) {
                    if (--snap_ctr == 0) { snap_ctr = p.snap_every; emit_record(); }   // S1
                }
                if (x1 > p.r_escape) finish(ST_ESCAPED);                         // B3
                else if (steps >= p.nsteps) finish(ST_MAXSTEPS);                 // B4
            }
        }
    }
}

// caller's table [5][n2][n1] (field-major) -> node-major A / B
__global__ void tab_pack_kernel(const double* __restrict__ src, long long nodes, double4* __restrict__ A, double* __restrict__ B) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nodes) return;
    A[k] = make_double4(src[k], src[nodes + k], src[2 * nodes + k], src[3 * nodes + k]);
    B[k] = src[4 * nodes + k];
}

}  // namespace geo
