// geo_rhs.cuh -- FP64 right-hand side of the geodesic equations in the paper's 3+1 variables.
//
// What is evaluated (eqs.(1)-(8); SURVEY/DESIGN "A2"):
//   H = 1/2 [ -(p_t - beta^k p_k)^2 / alpha^2 + gamma^{ij} p_i p_j ]          (eq.(4) with eq.(1))
// for the Kerr metric in 3+1 form, eq.(8) PAPER.md:97:
//   alpha^2 = rho^2 Delta / Sigma,  beta^phi = -omega = -2 M a r / Sigma,
//   gamma^{rr} = Delta / rho^2,  gamma^{thth} = 1 / rho^2,  gamma^{phph} = rho^2 / (Sigma sin^2 th),
//   rho^2 = r^2 + a^2 cos^2 th,  Delta = r^2 - 2 M r + a^2,  Sigma = (r^2+a^2)^2 - a^2 Delta sin^2 th
//   (PAPER.md:78-84), and Hamilton's equations (3) PAPER.md:60-63 with p_t(paper) = E, p_phi = L:
//   u^t     = (E - omega L) / alpha^2
//   dr/dtau = gamma^{rr} p_r,   dth/dtau = gamma^{thth} p_th,   dphi/dtau = gamma^{phph} L + omega u^t
//   dp_i/dtau = -1/2 (u^t)^2 d_i(alpha^2) - u^t L d_i(omega)
//               -1/2 ( d_i gamma^{rr} p_r^2 + d_i gamma^{thth} p_th^2 + d_i gamma^{phph} L^2 ),  i = r, th
//   dp_t/dtau = dp_phi/dtau = 0                                     (eqs.(13),(32) PAPER.md:116, 210)
// The metric derivatives are taken in closed form as logarithmic derivatives of alpha^2 and
// gamma^{phph} so that the four reciprocals 1/rho^2, 1/Delta, 1/Sigma, 1/sin^2 are the only divisions,
// and those come out of ONE reciprocal of the product.  Schwarzschild (a = 0) is the same system,
// eqs.(29)-(32) PAPER.md:203-211, and has its own shorter routine.
//
// Nothing here is shared with oracle/ (which uses the separable Carter form of the same H).
#pragma once
#include <cuda_runtime.h>

namespace geo {

// Constants of the sin/cos kernel.  They travel in the kernel parameters (constant bank), so that the
// DFMAs read them as constant operands: as literals the compiler re-materialises every coefficient with
// two MOV-immediates per use (ncu: 83 of 513 issued instructions per RK4 step).
struct TrigConsts {
    double two_over_pi, pio2_hi, pio2_lo;
    double s[6];   // sin y = y + y z (s0 + s1 z + ... + s5 z^5),  z = y^2
    double c[6];   // cos y = 1 - z/2 + z^2 (c0 + c1 z + ... + c5 z^5)
};

struct Hole {
    double M, a, a2, twoM, twoMa;
    TrigConsts tc;
};

// The twelve polynomial coefficients and the two-piece pi/2 are those of fdlibm's __kernel_sin / __kernel_cos
// (k_sin.c S1..S6, k_cos.c C1..C6; Sun Microsystems, freely distributable) and of its e_rem_pio2.c: a constant
// table, restated; the evaluation code around them is this file's own.
inline void fill_trig_consts(TrigConsts& t) {
    t.two_over_pi = 0.63661977236758134308;
    t.pio2_hi = 1.5707963267948966e+00;
    t.pio2_lo = 6.1232339957367660e-17;
    const double s[6] = {-1.66666666666666324348e-01, 8.33333333332248946124e-03, -1.98412698298579493134e-04,
                         2.75573137070700676789e-06, -2.50507602534068634195e-08, 1.58969099521155010221e-10};
    const double c[6] = {4.16666666666666019037e-02, -1.38888888888741095749e-03, 2.48015872894767294178e-05,
                         -2.75573143513906633035e-07, 2.08757232129817482790e-09, -1.13596475577881948265e-11};
    for (int i = 0; i < 6; ++i) { t.s[i] = s[i]; t.c[i] = c[i]; }
}

// d/dtau of (t, r, theta, phi, p_r, p_theta)
struct Deriv {
    double t, r, th, ph, pr, pth;
};

// 1/x for finite normal x, faithfully rounded (<= 1 ulp): MUFU.RCP64H seed (relative error
// <= 2^-20, measured: profiles/), then ONE cubic Newton correction y(1 + e + e^2), whose truncation
// error e^3 <= 2^-60 is far below the rounding of the final FMA.  No denormal / Inf slow path
// (garbage in, garbage out -- callers discard lanes whose inputs left the domain).
__device__ __forceinline__ double rcp_nr(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

// x = k pi/2 + y: returns sn = sin y, cs = cos y, odd = k & 1.  Cody-Waite reduction by pi/2 in two
// pieces (the first FMA is exact; |x| stays within a few pi on this path, so the neglected
// k * 1.5e-33 is far below an ulp of y), minimax polynomials on [-pi/4, pi/4] (fdlibm's degree-13 /
// degree-14 kernels, see fill_trig_consts; < 1 ulp), branch-free.
__device__ __forceinline__ void sincos_reduced(const TrigConsts& tc, double x, double& sn, double& cs, bool& odd) {
    const double magic = 6755399441055744.0;   // 1.5 * 2^52: adding it rounds to the nearest integer
    double kd = fma(x, tc.two_over_pi, magic);  // (zero low word: an immediate operand)
    odd = __double2loint(kd) & 1;
    kd -= magic;
    double y = fma(-kd, tc.pio2_hi, x);
    y = fma(-kd, tc.pio2_lo, y);
    const double z = y * y;
    double ps = fma(z, tc.s[5], tc.s[4]);
    ps = fma(ps, z, tc.s[3]);
    ps = fma(ps, z, tc.s[2]);
    ps = fma(ps, z, tc.s[1]);
    ps = fma(ps, z, tc.s[0]);
    double pc = fma(z, tc.c[5], tc.c[4]);
    pc = fma(pc, z, tc.c[3]);
    pc = fma(pc, z, tc.c[2]);
    pc = fma(pc, z, tc.c[1]);
    pc = fma(pc, z, tc.c[0]);
    sn = fma(y * z, ps, y);
    cs = fma(z, fma(z, pc, -0.5), 1.0);         // 1 - z/2 + z^2 pc(z), Horner: every FMA has one immediate operand
}

// s2 = sin^2 x and sc = sin x cos x -- the only trigonometric quantities the RHS needs (cos^2 enters
// as 1 - s2).  Odd quadrant: sin^2 x = cos^2 y, sin x cos x = -sin y cos y (sign flip on the integer pipe).
__device__ __forceinline__ void sin2_sincos(const TrigConsts& tc, double x, double& s2, double& sc) {
    double sn, cs;
    bool odd;
    sincos_reduced(tc, x, sn, cs, odd);
    const double S = odd ? cs : sn;
    s2 = S * S;
    const double p = sn * cs;
    sc = __hiloint2double(__double2hiint(p) ^ (odd ? 0x80000000 : 0), __double2loint(p));
}

// (S, C) = (sin x, cos x) up to ONE COMMON sign -- all that s2 = S^2 and sc = S C need, and the
// rotation below preserves it.  Used once per RK4 step, at the step's base point.
__device__ __forceinline__ void sincos_common_sign(const TrigConsts& tc, double x, double& S, double& C) {
    double sn, cs;
    bool odd;
    sincos_reduced(tc, x, sn, cs, odd);
    S = odd ? cs : sn;   // x = k pi/2 + y, k odd: sin = +-cos y, cos = -+sin y
    const double ns = __hiloint2double(__double2hiint(sn) ^ 0x80000000, __double2loint(sn));
    C = odd ? ns : cs;
}

// sin^2 and sin cos at theta + d from (S, C) at theta -- the RK4 stage points sit at
// d = (h/2 or h) * dtheta/dtau from the step's base point, so the angle-addition theorem with short Taylor
// kernels for (sin d, cos d - 1) replaces a full sin/cos evaluation: 13 FP64 instructions instead of 22,
// and no branch, so the four RHS evaluations of a step stay in ONE basic block for the scheduler.
// For |d| < 2^-7 the kernels are exact to rounding (truncation d^7/5040 < 3.5e-19 relative for sin,
// d^8/40320 < 3e-22 for cos).  A larger d (only next to the horizon, or with a coarse h) sets `coarse`;
// the caller then discards the step's sum and recomputes it with full sin/cos evaluations
// (rk4_sum_full).  The decision is per lane, on the integer pipe: a particle's arithmetic never depends
// on its neighbours.  The leading coefficients of the minimax kernels stand in for -1/6, 1/120, 1/24,
// -1/720: they differ by < 1e-13 relative, which the factors d^2 <= 6e-5 push below 1e-17.
__device__ __forceinline__ void stage_trig(const TrigConsts& tc, double S, double C, double d,
                                           double& s2, double& sc, unsigned& dmax) {
    const double d2 = d * d;
    dmax = max(dmax, (unsigned)__double2hiint(d2));      // d^2 >= 2^-14 <=> |d| >= 2^-7; a NaN ranks above both (unsigned)
    const double sd = fma(d * d2, fma(d2, tc.s[1], tc.s[0]), d);            // sin d
    const double cm = d2 * fma(fma(d2, tc.c[1], tc.c[0]), d2, -0.5);        // cos d - 1
    const double s1 = fma(S, cm, fma(C, sd, S));                            // sin(theta + d)
    const double c1 = fma(C, cm, fma(-S, sd, C));                           // cos(theta + d)
    s2 = s1 * s1;
    sc = s1 * c1;
}

// Kerr, eq.(8) variables.  (r, th, pr, pth) evolving; E, L constants of motion.
//
// With W = E + beta^phi L = E - omega L,  u^t = W / alpha^2,  q1 = alpha^2 (u^t)^2 = W u^t,
// G = gamma^{phph} L^2,  B = q1 + G,  Krho = gamma^{rr} p_r^2 + gamma^{thth} p_th^2,
// the momentum equations of the header, with the closed-form derivatives
//   d_r ln alpha^2   = 2r/rho^2 + 2(r-M)/Delta - d_r Sigma / Sigma,   d_th ln alpha^2 = 2 a^2 s c (Delta/Sigma - 1/rho^2)
//   d_r omega        = (2Ma - omega d_r Sigma)/Sigma,                 d_th omega      = 2 a^2 s c Delta omega / Sigma
//   d_r gamma^{rr}   = 2(r-M)/rho^2 - 2r gamma^{rr}/rho^2,            d_th gamma^{rr} = 2 a^2 s c gamma^{rr}/rho^2
//   d_r gamma^{thth} = -2r/rho^4,                                     d_th gamma^{thth} = 2 a^2 s c / rho^4
//   d_r ln gamma^{phph} = 2r/rho^2 - d_r Sigma/Sigma,                 d_th ln gamma^{phph} = d_th ln alpha^2 ... - 2 c/s
//   d_r Sigma = 4 r (r^2+a^2) - 2 a^2 (r-M) s^2,                      d_th Sigma = -2 a^2 Delta s c
// collect (terms in d_r Sigma / Sigma, in 1/rho^2, in (r-M)) into
//   X = B + 2 u^t L omega,   Z = X / Sigma,   Y = (Krho - B) / rho^2
//   dp_r/dtau  = r Y + 2 r (r^2+a^2) Z - (r-M) [ a^2 s^2 Z + q1/Delta + p_r^2/rho^2 ] - u^t L 2Ma/Sigma
//   dp_th/dtau = s c { G / s^2 - a^2 (Delta Z + Y) }
// (checked against the mpmath differentiation of H that pins the oracle: tests/test_oracle_pins.py
// runs on the oracle; tests/test_gpu_parity.py compares the two).  58 FP64 instructions + sin/cos.
__device__ __forceinline__ void rhs_kerr(const Hole& bh, double r, double s2, double sc, double pr, double pth,
                                         double E, double L, Deriv& d) {
    const double r2 = r * r;
    const double A = r2 + bh.a2;                       // r^2 + a^2
    const double a2s2 = bh.a2 * s2;
    const double rho2 = A - a2s2;                      // r^2 + a^2 cos^2
    const double Delta = fma(-bh.twoM, r, A);
    const double Sigma = fma(A, A, -(a2s2 * Delta));
    // one reciprocal gives 1/rho^2, 1/Delta, 1/Sigma, 1/sin^2 (issue slots are the bound: a second
    // MUFU + zero-extension costs as much as the two multiplications that split the product)
    const double P1 = rho2 * Delta, P2 = Sigma * s2;
    const double iP = rcp_nr(P1 * P2);
    const double iP1 = iP * P2;                        // 1/(rho^2 Delta)
    const double iP2 = iP * P1;                        // 1/(Sigma sin^2)
    const double irho = iP1 * Delta, iDel = iP1 * rho2;
    const double iSig = iP2 * s2, is2 = iP2 * Sigma;
    // lapse, shift, 3-metric (eq.(8))
    const double mS = bh.twoMa * iSig;                 // 2Ma / Sigma
    const double omega = mS * r;                       // -beta^phi
    const double W = fma(-omega, L, E);                // E + beta^phi L
    const double ut = (W * Sigma) * iP1;               // W / alpha^2
    const double q1 = W * ut;                          // alpha^2 (u^t)^2
    const double gL = (rho2 * iP2) * L;                // gamma^{phph} L
    const double G = gL * L;
    const double pri = pr * irho;                      // p_r / rho^2
    d.t = ut;
    d.r = Delta * pri;                                 // gamma^{rr} p_r
    d.th = irho * pth;                                 // gamma^{thth} p_th
    d.ph = fma(omega, ut, gL);
    const double B = q1 + G;
    const double KB = fma(d.r, pr, fma(d.th, pth, -B));   // Krho - B
    const double Y = irho * KB;
    const double u1 = (ut * L) * mS;                   // u^t L 2Ma / Sigma
    const double r2x = r + r;
    const double Z = iSig * fma(u1, r2x, B);           // X / Sigma
    const double br = fma(a2s2, Z, fma(q1, iDel, pr * pri));
    const double rmM = r - bh.M;
    d.pr = fma(-rmM, br, fma(r2x * A, Z, fma(r, Y, -u1)));
    d.pth = sc * fma(-bh.a2, fma(Delta, Z, Y), G * is2);
}

// Schwarzschild: alpha^2 = 1 - 2M/r = gamma^{rr}, gamma^{thth} = 1/r^2, gamma^{phph} = 1/(r^2 sin^2),
// beta^i = 0 -- eq.(8) at a = 0; the result is eqs.(29)-(32) PAPER.md:203-211.
__device__ __forceinline__ void rhs_schwarzschild(const Hole& bh, double r, double s2, double sc, double pr,
                                                  double pth, double E, double L, Deriv& d) {
    const double r2 = r * r;
    const double Delta = fma(-bh.twoM, r, r2);         // r^2 alpha^2
    const double P2 = r2 * s2;
    const double iP = rcp_nr(Delta * P2);
    const double iDel = iP * P2;                       // 1/Delta
    const double iP2 = iP * Delta;                     // gamma^{phph} = 1/(r^2 sin^2)
    const double ir2 = iP2 * s2;                       // gamma^{thth}
    const double is2 = iP2 * r2;
    const double ut = (E * r2) * iDel;                 // E / alpha^2
    const double gL = iP2 * L;
    d.t = ut;
    d.r = (Delta * ir2) * pr;
    d.th = ir2 * pth;
    d.ph = gL;
    const double G = gL * L;                           // gamma^{phph} L^2
    // -1/2 (u^t)^2 d_r alpha^2 - 1/2 d_r gamma^{rr} p_r^2 = -(M/r^2)(ut^2 + pr^2);
    // -1/2 (d_r gamma^{thth} pth^2 + d_r gamma^{phph} L^2) = (gthth pth^2 + G)/r
    const double Mr2 = bh.M * ir2;
    const double cen = fma(ir2, pth * pth, G) * (r * ir2);
    d.pr = fma(-Mr2, fma(ut, ut, pr * pr), cen);
    d.pth = (G * sc) * is2;                            // -1/2 d_th gamma^{phph} L^2
}

template <bool KERR>
__device__ __forceinline__ void rhs(const Hole& bh, double r, double s2, double sc, double pr, double pth,
                                    double E, double L, Deriv& d) {
    if (KERR) rhs_kerr(bh, r, s2, sc, pr, pth, E, L, d);
    else rhs_schwarzschild(bh, r, s2, sc, pr, pth, E, L, d);
}

// --- cold-path helpers: IEEE division / sqrt / libdevice sincos, called once per particle ---------

// E = alpha sqrt(kappa + gamma^{ij} u_i u_j) - beta^phi u_phi: the mass shell eq.(5)
// solved for p_t in the variables of eq.(1), future-directed root.
__device__ __noinline__ double energy_3p1(const Hole& bh, double r, double th, double pr, double pth,
                                          double L, double kappa) {
    double s, c;
    sincos(th, &s, &c);
    const double s2 = s * s;
    const double A = r * r + bh.a2;
    const double rho2 = r * r + bh.a2 * c * c;
    const double Delta = A - bh.twoM * r;
    const double Sigma = A * A - bh.a2 * Delta * s2;
    const double alpha2 = rho2 * Delta / Sigma;
    const double omega = bh.twoMa * r / Sigma;
    const double g = (Delta * pr * pr + pth * pth) / rho2 + rho2 * L * L / (Sigma * s2);
    return sqrt(alpha2 * (kappa + g)) + omega * L;
}

// sin x and cos x with their true signs, for |x| up to ~2^20 (phi of a long orbit): the reduction of sincos_reduced,
// then the quadrant k mod 4 from the two low bits of k (integer pipe).  Absolute error ~1e-16 (1 + |x| 2^-52).
__device__ __forceinline__ void sincos_full(const TrigConsts& tc, double x, double& sn, double& cs) {
    const double magic = 6755399441055744.0;
    const double kd0 = fma(x, tc.two_over_pi, magic);
    const int q = __double2loint(kd0);
    const double kd = kd0 - magic;
    double y = fma(-kd, tc.pio2_hi, x);
    y = fma(-kd, tc.pio2_lo, y);
    const double z = y * y;
    double ps = fma(z, tc.s[5], tc.s[4]);
    ps = fma(ps, z, tc.s[3]);
    ps = fma(ps, z, tc.s[2]);
    ps = fma(ps, z, tc.s[1]);
    ps = fma(ps, z, tc.s[0]);
    double pc = fma(z, tc.c[5], tc.c[4]);
    pc = fma(pc, z, tc.c[3]);
    pc = fma(pc, z, tc.c[2]);
    pc = fma(pc, z, tc.c[1]);
    pc = fma(pc, z, tc.c[0]);
    const double s0 = fma(y * z, ps, y);
    const double c0 = fma(z, fma(z, pc, -0.5), 1.0);
    const double a = (q & 1) ? c0 : s0, b = (q & 1) ? s0 : c0;      // k odd: sin = +-cos y, cos = -+sin y
    const int ssn = (q & 2) ? 0x80000000 : 0;                       // k = 2, 3: sin changes sign
    const int scs = ((q + 1) & 2) ? 0x80000000 : 0;                 // k = 1, 2: cos changes sign
    sn = __hiloint2double(__double2hiint(a) ^ ssn, __double2loint(a));
    cs = __hiloint2double(__double2hiint(b) ^ scs, __double2loint(b));
}

// sqrt(x) for finite normal x > 0, faithfully rounded: MUFU.RSQ64H seed (relative error ~2^-20), one coupled
// Goldschmidt step for (sqrt x, 1/(2 sqrt x)) and a final residual correction.  No special-case path.
__device__ __forceinline__ double sqrt_nr(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double g = x * y, h = 0.5 * y;
    const double r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    return fma(fma(-g, g, x), h, g);
}

// Boyer-Lindquist -> Cartesian, eq.(7) PAPER.md:88-93 -- the paper's output format, fused into the
// snapshot writer.  Inlined and branch-free (~60 FP64 instructions): with a record EVERY step -- the
// paper's own mode -- the conversion runs once per RK4 step, and the round-1 version (an out-of-line routine built on
// libdevice's sincos and sqrt) cost more than the step's own trigonometry.
__device__ __forceinline__ void cartesian_eq7(const TrigConsts& tc, double a2, double r, double th, double ph,
                                              double& x, double& y, double& z) {
    double st, ct, sp, cp;
    sincos_full(tc, th, st, ct);
    sincos_full(tc, ph, sp, cp);
    const double w = sqrt_nr(fma(r, r, a2)) * st;
    x = w * cp;
    y = w * sp;
    z = r * ct;
}

// |2H + kappa| with 2H = -alpha^2 (u^t)^2 + gamma^{ij} p_i p_j (B7 "health").
__device__ __noinline__ double health_3p1(const Hole& bh, double r, double th, double pr, double pth,
                                          double E, double L, double kappa) {
    double s, c;
    sincos(th, &s, &c);
    const double s2 = s * s;
    const double A = r * r + bh.a2;
    const double rho2 = r * r + bh.a2 * c * c;
    const double Delta = A - bh.twoM * r;
    const double Sigma = A * A - bh.a2 * Delta * s2;
    const double alpha2 = rho2 * Delta / Sigma;
    const double omega = bh.twoMa * r / Sigma;
    const double W = E - omega * L;
    const double twoH = -W * W / alpha2 + (Delta * pr * pr + pth * pth) / rho2 + rho2 * L * L / (Sigma * s2);
    return fabs(twoH + kappa);
}

}  // namespace geo
