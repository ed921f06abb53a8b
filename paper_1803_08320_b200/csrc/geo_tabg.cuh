// geo_tabg.cuh -- SURVEY 8(f).3, second part (reading T6): fixed-step RK4 geodesics through a GENERAL
// stationary, axisymmetric, numerically given 3+1 metric -- all ten functions of line element (1):
// lapse alpha, shift (beta^1, beta^2, beta^3), spatial metric gamma_11, gamma_12, gamma_13, gamma_22, gamma_23,
// gamma_33 on a uniform (x^1, x^2) grid (x^3 = phi is the symmetry direction).  No circularity and no diagonal
// 3-metric is assumed, so horizon-penetrating coordinates (Kerr-Schild: beta^r != 0, gamma_r phi != 0) are inside its
// scope -- the paper's stated purpose of the 3+1 form is "future support to numerical metrics".
//
//   H = 1/2 [ -W^2/alpha^2 + gamma^{ij} p_i p_j ],  p = (p_1, p_2, L),  W = E + beta^k p_k,  u^t = W/alpha^2,  V^i = gamma^{ij} p_j
//   dt/dtau = u^t,   dx^i/dtau = V^i - beta^i u^t,
//   dp_k/dtau = -alpha (u^t)^2 d_k alpha + u^t p_j d_k beta^j + 1/2 V^a V^b d_k gamma_ab   (k = 1, 2),   dL/dtau = dE/dtau = 0
//
// Interpolant, its exact gradient, domain rule, stepper, stop rules and events: those of geo_tab.cuh (readings T2, T4, T5).
// Table layout on the device (built once by tabg_pack_kernel from the caller's [10][n2][n1]): node-major records of
// 12 doubles = 96 B (10 fields + 2 pad) -> three 256-bit loads per node, 48 per stencil and lane.
// v1 (GEO_FLAG_TAB_GATHER) gathers the 4 x 4 stencil on every evaluation: L1-wavefront-bound (ncu: 89 % of the L1
// data-pipe peak, FP64 pipe 19 %).  v2 (default) keeps the stencil of the lane's current cell -- 160 doubles = 1.25 KB
// per lane -- in shared memory, column-major [160][32] per 32-lane CTA (40 KB; five CTAs per SM), and refills it only when
// the cell index changes (a particle stays in a cell for tens of evaluations).  Same arithmetic, same bits.
#pragma once
#include "geo_tab.cuh"

namespace geo {

constexpr int kTabgFields = 10;
constexpr int kTabgStride = 12;      // doubles per node record (96 B: 32-byte aligned)

struct TabgMetric {
    const double* G;   // [n2][n1][12]
    int n1, n2;
    double x1_0, d1, inv_d1, x2_0, d2, inv_d2;
};

struct TabgParams {
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
    TabgMetric m;
};

struct TabgFields {
    double v[kTabgFields], g1[kTabgFields], g2[kTabgFields];   // value, d/dx^1, d/dx^2
};

// Interpolated fields and gradients at (x1, x2); false outside the domain (values then finite garbage of a clamped cell).
__device__ __forceinline__ bool tabg_fields(const TabgMetric& m, double x1, double x2, TabgFields& F) {
    int i, j;
    double s1, s2;
    const bool in1 = tab_cell(x1, m.x1_0, m.d1, m.inv_d1, m.n1, i, s1);
    const bool in2 = tab_cell(x2, m.x2_0, m.d2, m.inv_d2, m.n2, j, s2);
    double w1[4], dw1[4], w2[4], dw2[4];
    keys_weights(s1, m.inv_d1, w1, dw1);
    keys_weights(s2, m.inv_d2, w2, dw2);
#pragma unroll
    for (int f = 0; f < kTabgFields; ++f) F.v[f] = F.g1[f] = F.g2[f] = 0.0;
    const long long base = ((long long)(j - 1) * m.n1 + (i - 1)) * kTabgStride;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const double4* row = reinterpret_cast<const double4*>(m.G + base + (long long)b * m.n1 * kTabgStride);
        double c[4][kTabgStride];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                const double4 t = ldg256(row + a * 3 + q);
                c[a][4 * q] = t.x; c[a][4 * q + 1] = t.y; c[a][4 * q + 2] = t.z; c[a][4 * q + 3] = t.w;
            }
        }
#pragma unroll
        for (int f = 0; f < kTabgFields; ++f) {
            const double rv = fma(w1[3], c[3][f], fma(w1[2], c[2][f], fma(w1[1], c[1][f], w1[0] * c[0][f])));
            const double rd = fma(dw1[3], c[3][f], fma(dw1[2], c[2][f], fma(dw1[1], c[1][f], dw1[0] * c[0][f])));
            F.v[f] = fma(w2[b], rv, F.v[f]);
            F.g1[f] = fma(w2[b], rd, F.g1[f]);
            F.g2[f] = fma(dw2[b], rv, F.g2[f]);
        }
    }
    return in1 & in2;
}

// CACHE variant of tabg_fields: the stencil comes from the lane's shared-memory column `col` (stride `cs` doubles
// between consecutive elements), refilled from the table when the cell (i, j) differs from (ci, cj).
__device__ __forceinline__ bool tabg_fields_cached(const TabgMetric& m, double x1, double x2, TabgFields& F, int& ci, int& cj,
                                                   double* col, int cs) {
    int i, j;
    double s1, s2;
    const bool in1 = tab_cell(x1, m.x1_0, m.d1, m.inv_d1, m.n1, i, s1);
    const bool in2 = tab_cell(x2, m.x2_0, m.d2, m.inv_d2, m.n2, j, s2);
    if (i != ci || j != cj) {
        const long long base = ((long long)(j - 1) * m.n1 + (i - 1)) * kTabgStride;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double4* row = reinterpret_cast<const double4*>(m.G + base + (long long)b * m.n1 * kTabgStride);
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const double4 t0 = ldg256(row + a * 3), t1 = ldg256(row + a * 3 + 1), t2 = ldg256(row + a * 3 + 2);
                double* e = col + (size_t)((b * 4 + a) * kTabgFields) * cs;
                e[0] = t0.x; e[cs] = t0.y; e[2 * cs] = t0.z; e[3 * cs] = t0.w;
                e[4 * cs] = t1.x; e[5 * cs] = t1.y; e[6 * cs] = t1.z; e[7 * cs] = t1.w;
                e[8 * cs] = t2.x; e[9 * cs] = t2.y;
            }
        }
        ci = i;
        cj = j;
    }
    double w1[4], dw1[4], w2[4], dw2[4];
    keys_weights(s1, m.inv_d1, w1, dw1);
    keys_weights(s2, m.inv_d2, w2, dw2);
#pragma unroll
    for (int f = 0; f < kTabgFields; ++f) F.v[f] = F.g1[f] = F.g2[f] = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
#pragma unroll
        for (int f = 0; f < kTabgFields; ++f) {
            const double c0 = col[(size_t)((b * 4 + 0) * kTabgFields + f) * cs], c1 = col[(size_t)((b * 4 + 1) * kTabgFields + f) * cs],
                         c2 = col[(size_t)((b * 4 + 2) * kTabgFields + f) * cs], c3 = col[(size_t)((b * 4 + 3) * kTabgFields + f) * cs];
            const double rv = fma(w1[3], c3, fma(w1[2], c2, fma(w1[1], c1, w1[0] * c0)));
            const double rd = fma(dw1[3], c3, fma(dw1[2], c2, fma(dw1[1], c1, dw1[0] * c0)));
            F.v[f] = fma(w2[b], rv, F.v[f]);
            F.g1[f] = fma(w2[b], rd, F.g1[f]);
            F.g2[f] = fma(dw2[b], rv, F.g2[f]);
        }
    }
    return in1 & in2;
}

constexpr int kTabgCacheBlock = 32;                                  // lanes per CTA of the cached variant
constexpr int kTabgCacheRows = 16 * kTabgFields;                     // doubles per lane

struct TabgAux {
    double V1, V2, V3, W, ut, gpp;
};

// gamma^{ij} p_j by the adjugate of the symmetric 3 x 3 matrix (one reciprocal of the determinant), W, u^t
__device__ __forceinline__ TabgAux tabg_aux(const double* v, double p1, double p2, double L, double E) {
    const double a = v[4], b = v[5], c = v[6], d = v[7], e = v[8], g = v[9];
    const double c11 = fma(d, g, -e * e), c12 = fma(c, e, -b * g), c13 = fma(b, e, -c * d);
    const double c22 = fma(a, g, -c * c), c23 = fma(b, c, -a * e), c33 = fma(a, d, -b * b);
    const double idet = rcp_nr(fma(a, c11, fma(b, c12, c * c13)));
    TabgAux A;
    A.V1 = idet * fma(c11, p1, fma(c12, p2, c13 * L));
    A.V2 = idet * fma(c12, p1, fma(c22, p2, c23 * L));
    A.V3 = idet * fma(c13, p1, fma(c23, p2, c33 * L));
    A.gpp = fma(A.V1, p1, fma(A.V2, p2, A.V3 * L));
    A.W = fma(v[1], p1, fma(v[2], p2, fma(v[3], L, E)));
    A.ut = A.W * rcp_nr(v[0] * v[0]);
    return A;
}

__device__ __forceinline__ void tabg_rhs(const TabgFields& F, double p1, double p2, double E, double L, TabDeriv& d) {
    const TabgAux A = tabg_aux(F.v, p1, p2, L, E);
    d.t = A.ut;
    d.x1 = fma(-F.v[1], A.ut, A.V1);
    d.x2 = fma(-F.v[2], A.ut, A.V2);
    d.ph = fma(-F.v[3], A.ut, A.V3);
    const double q = -F.v[0] * A.ut * A.ut;
    const double h11 = 0.5 * A.V1 * A.V1, h22 = 0.5 * A.V2 * A.V2, h33 = 0.5 * A.V3 * A.V3;
    const double h12 = A.V1 * A.V2, h13 = A.V1 * A.V3, h23 = A.V2 * A.V3;
    const double up1 = A.ut * p1, up2 = A.ut * p2, upL = A.ut * L;
#define GEO_TABG_DP(g)                                                                                                 \
    fma(q, g[0], fma(up1, g[1], fma(up2, g[2], fma(upL, g[3], fma(h11, g[4], fma(h12, g[5], fma(h13, g[6],               \
        fma(h22, g[7], fma(h23, g[8], h33 * g[9])))))))))
    d.p1 = GEO_TABG_DP(F.g1);
    d.p2 = GEO_TABG_DP(F.g2);
#undef GEO_TABG_DP
}

__device__ __noinline__ bool tabg_fields_cold(const TabgMetric& m, double x1, double x2, TabgFields& F) {
    return tabg_fields(m, x1, x2, F);
}

template <bool PLAIN, bool CACHE, bool SNAP>
__global__ void __launch_bounds__(CACHE ? kTabgCacheBlock : kTabBlock, CACHE ? 5 : 2) geo_tabg_rk4_kernel(const __grid_constant__ TabgParams p) {
    extern __shared__ __align__(16) double tabg_smem[];              // CACHE: [160][blockDim.x]
    double* const col = tabg_smem + threadIdx.x;
    const int cs = (int)blockDim.x;
    int ci = -1, cj = -1;                                            // cell whose stencil the column holds
    const unsigned lane = threadIdx.x & 31u;
    const TabgMetric& m = p.m;
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
            TabgFields F;
            double hv = qnan;
            if (tabg_fields_cold(m, x1, x2, F) && (__double2hiint(E) & 0x7ff00000) != 0x7ff00000) {
                const TabgAux A = tabg_aux(F.v, p1, p2, L, E);
                hv = fabs(-(A.W * A.W) / (F.v[0] * F.v[0]) + A.gpp + p.kappa);
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
        TabgFields F;
        if (!tabg_fields_cold(m, x1, x2, F)) { finish(ST_OUTSIDE); return; }     // T4 on y0
        const TabgAux A = tabg_aux(F.v, p1, p2, L, 0.0);                         // mass shell (5): A.W = beta^k p_k here
        E = fma(F.v[0], sqrt(p.kappa + A.gpp), -A.W);
        if ((__double2hiint(E) & 0x7ff00000) == 0x7ff00000) { finish(ST_NUMERIC); return; }
        if (SNAP) emit_record();                                                 // S1: slot 0 = y0
        if (x1 > p.r_escape) { finish(ST_ESCAPED); return; }
        if (p.nsteps == 0) { finish(ST_MAXSTEPS); return; }
        tabg_rhs(F, p1, p2, E, L, k1);
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

        // --- one RK4 step: the four evaluations (stage points 2-4, end point) through ONE copy of the evaluator ------
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
                kahan<PLAIN>(t, ct, p.h_sixth, at, nt, dt);
                kahan<PLAIN>(x1, c1, p.h_sixth, a1, n1, d1);
                kahan<PLAIN>(x2, c2, p.h_sixth, a2, n2, d2);
                kahan<PLAIN>(ph, cph, p.h_sixth, aph, nph, dph);
                kahan<PLAIN>(p1, cp1, p.h_sixth, ap1, np1, dp1);
                kahan<PLAIN>(p2, cp2, p.h_sixth, ap2, np2, dp2);
                e1 = n1; e2 = n2; ep1 = np1; ep2 = np2;
                fin6 = all_finite6(nt, n1, n2, nph, np1, np2);
            }
            TabgFields F;
            const bool in = CACHE ? tabg_fields_cached(m, e1, e2, F, ci, cj, col, cs) : tabg_fields(m, e1, e2, F);
            if (!ev) ev = !(e1 >= p.r_capture) ? ST_CAPTURED : (!fin6 ? ST_NUMERIC : (!in ? ST_OUTSIDE : 0));
            tabg_rhs(F, ep1, ep2, E, L, d);
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

// caller's table [10][n2][n1] (field-major) -> node-major records of 12 doubles
__global__ void tabg_pack_kernel(const double* __restrict__ src, long long nodes, double* __restrict__ G) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nodes) return;
#pragma unroll
    for (int f = 0; f < kTabgFields; ++f) G[k * kTabgStride + f] = src[(long long)f * nodes + k];
    G[k * kTabgStride + 10] = 0.0;
    G[k * kTabgStride + 11] = 0.0;
}

}  // namespace geo
