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

struct Hole {
    double M, a, a2, twoM, twoMa, twoa2;
};

// d/dtau of (t, r, theta, phi, p_r, p_theta)
struct Deriv {
    double t, r, th, ph, pr, pth;
};

// 1/x for finite normal x, <= 1 ulp: MUFU.RCP64H seed (rel. err ~2^-20), one cubic and one
// quadratic Newton correction, no denormal / Inf slow path (garbage in, garbage out -- callers
// discard lanes whose inputs left the domain).
__device__ __forceinline__ double rcp_nr(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    double t = fma(e, e, e);
    y = fma(y, t, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

// S = +-sin(x), C = +-cos(x) up to ONE COMMON sign (the RHS only uses S^2, C^2 and S*C, all even
// under (S,C) -> (-S,-C)).  Cody-Waite reduction by pi/2 in three pieces, minimax polynomials on
// [-pi/4, pi/4] (the classical degree-13 / degree-14 kernels, max err < 1 ulp), branch-free.
__device__ __forceinline__ void sincos_even(double x, double& S, double& C) {
    const double magic = 6755399441055744.0;  // 1.5 * 2^52: adds round-to-nearest-integer
    double kd = fma(x, 0.63661977236758134308, magic);
    const int q = __double2loint(kd);
    kd -= magic;
    double y = fma(-kd, 1.5707963267948966e+00, x);
    y = fma(-kd, 6.1232339957367660e-17, y);
    y = fma(-kd, -1.4973849048591698e-33, y);
    const double z = y * y;
    double ps = fma(z, 1.58969099521155010221e-10, -2.50507602534068634195e-08);
    ps = fma(ps, z, 2.75573137070700676789e-06);
    ps = fma(ps, z, -1.98412698298579493134e-04);
    ps = fma(ps, z, 8.33333333332248946124e-03);
    ps = fma(ps, z, -1.66666666666666324348e-01);
    double pc = fma(z, -1.13596475577881948265e-11, 2.08757232129817482790e-09);
    pc = fma(pc, z, -2.75573143513906633035e-07);
    pc = fma(pc, z, 2.48015872894767294178e-05);
    pc = fma(pc, z, -1.38888888888741095749e-03);
    pc = fma(pc, z, 4.16666666666666019037e-02);
    const double sn = fma(y * z, ps, y);
    const double cs = fma(z * z, pc, fma(z, -0.5, 1.0));
    const bool odd = q & 1;
    S = odd ? cs : sn;   // x = k pi/2 + y, k odd: sin = +-cos y, cos = -+sin y
    C = odd ? -sn : cs;
}

// Kerr, eq.(8) variables.  (r, th, pr, pth) evolving; E, L constants of motion.
__device__ __forceinline__ void rhs_kerr(const Hole& bh, double r, double th, double pr, double pth,
                                         double E, double L, Deriv& d) {
    double S, C;
    sincos_even(th, S, C);
    const double s2 = S * S, c2 = C * C, sc = S * C;
    const double r2 = r * r;
    const double A = r2 + bh.a2;                       // r^2 + a^2
    const double rho2 = fma(bh.a2, c2, r2);
    const double Delta = fma(-bh.twoM, r, A);
    const double a2D = bh.a2 * Delta;
    const double Sigma = fma(A, A, -(a2D * s2));
    // one reciprocal for 1/rho^2, 1/Delta, 1/Sigma, 1/sin^2
    const double P1 = rho2 * Delta, P2 = Sigma * s2;
    const double iP = rcp_nr(P1 * P2);
    const double iP1 = iP * P2, iP2 = iP * P1;         // 1/(rho^2 Delta), 1/(Sigma sin^2)
    const double irho = iP1 * Delta, iDel = iP1 * rho2;
    const double iSig = iP2 * s2, is2 = iP2 * Sigma;
    // lapse, shift, 3-metric (eq.(8))
    const double omega = (bh.twoMa * r) * iSig;        // -beta^phi
    const double W = fma(-omega, L, E);                // E + beta^phi L
    const double ut = (W * Sigma) * iP1;               // W / alpha^2
    const double grr = Delta * irho;                   // gamma^{rr}
    const double gL = (rho2 * iP2) * L;                // gamma^{phph} L
    const double G = gL * L;
    d.t = ut;
    d.r = grr * pr;
    d.th = irho * pth;
    d.ph = fma(omega, ut, gL);
    // closed-form derivatives
    const double rmM = r - bh.M;
    const double Sig_r = fma(4.0 * r, A, -2.0 * ((bh.a2 * rmM) * s2));   // d_r Sigma
    const double Tr = fma(r + r, irho, -(Sig_r * iSig));                 // d_r ln gamma^{phph}
    const double tsc = bh.twoa2 * sc;                                    // 2 a^2 sin cos
    const double Tth = tsc * fma(Delta, iSig, -irho);                    // d_th ln alpha^2
    const double pr2 = pr * pr;
    const double K = (fma(Delta, pr2, pth * pth) * irho) * irho;         // (grr pr^2 + gthth pth^2)/rho^2
    const double q1 = W * ut;                                            // alpha^2 (u^t)^2
    const double hB = 0.5 * (q1 + G);
    const double dw_r = fma(-omega, Sig_r, bh.twoMa) * iSig;             // d_r omega
    const double dw_th = ((omega * tsc) * Delta) * iSig;                 // d_th omega
    const double utL = ut * L;
    // d_r ln alpha^2 = Tr + 2 (r-M)/Delta ; d_r gamma^{rr} = 2 (r-M)/rho^2 - 2 r gamma^{rr}/rho^2
    double x = hB * Tr;
    x = fma(rmM, fma(q1, iDel, irho * pr2), x);
    x = fma(utL, dw_r, x);
    d.pr = fma(r, K, -x);
    // d_th ln gamma^{phph} = Tth - 2 cos/sin ; d_th gamma^{rr,thth} = 2 a^2 sin cos (.)/rho^4
    double w = hB * Tth;
    w = fma(utL, dw_th, w);
    w = fma(0.5 * tsc, K, w);
    d.pth = fma(G * sc, is2, -w);
}

// Schwarzschild: alpha^2 = 1 - 2M/r = gamma^{rr}, gamma^{thth} = 1/r^2, gamma^{phph} = 1/(r^2 sin^2),
// beta^i = 0 -- eq.(8) at a = 0; the result is eqs.(29)-(32) PAPER.md:203-211.
__device__ __forceinline__ void rhs_schwarzschild(const Hole& bh, double r, double th, double pr,
                                                  double pth, double E, double L, Deriv& d) {
    double S, C;
    sincos_even(th, S, C);
    const double s2 = S * S;
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
    d.pth = (G * (S * C)) * is2;                       // -1/2 d_th gamma^{phph} L^2
}

template <bool KERR>
__device__ __forceinline__ void rhs(const Hole& bh, double r, double th, double pr, double pth,
                                    double E, double L, Deriv& d) {
    if (KERR) rhs_kerr(bh, r, th, pr, pth, E, L, d);
    else rhs_schwarzschild(bh, r, th, pr, pth, E, L, d);
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
