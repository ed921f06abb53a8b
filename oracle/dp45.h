// dp45.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (part of the CPU oracle; see geo_oracle.cpp).
//
// The Dormand-Prince 5(4) pair used by the oracle's adaptive paths (geo_oracle.cpp: analytic metrics;
// geo_tab_oracle.cpp: tabulated metric): Butcher tableau (Dormand & Prince, J. Comput. Appl. Math. 6 (1980) 19,
// table 2), the controller's parameters, and the continuous extension (readings A1-A3).  Pinned by
// tests/test_oracle_adaptive.py through oracle_dp45_tableau / oracle_dp45_dense_weights.
#pragma once

namespace {

struct DP45 {
    static constexpr int S = 7;
    const long double c[S] = {0.0L, 1.0L / 5, 3.0L / 10, 4.0L / 5, 8.0L / 9, 1.0L, 1.0L};
    const long double a[S][S] = {
        {0},
        {1.0L / 5},
        {3.0L / 40, 9.0L / 40},
        {44.0L / 45, -56.0L / 15, 32.0L / 9},
        {19372.0L / 6561, -25360.0L / 2187, 64448.0L / 6561, -212.0L / 729},
        {9017.0L / 3168, -355.0L / 33, 46732.0L / 5247, 49.0L / 176, -5103.0L / 18656},
        {35.0L / 384, 0.0L, 500.0L / 1113, 125.0L / 192, -2187.0L / 6784, 11.0L / 84}};
    // 5th-order weights = last row of a; embedded 4th-order weights:
    const long double b4[S] = {5179.0L / 57600, 0.0L, 7571.0L / 16695, 393.0L / 640, -92097.0L / 339200,
                               187.0L / 2100, 1.0L / 40};
};

struct AdaptiveCtl { double h0, rtol, atol, h_min, tau_end, snap_dtau; };   // tau_end = +inf: no final time; snap_dtau = 0: no records

// Dense output of the pair (reading A3): the continuous extension of DOPRI5 as implemented in Hairer's dopri5
// ("contd5"; Hairer, Norsett & Wanner, Solving ODEs I, sec. II.6), fourth-order accurate on the whole step:
//   y(tau_n + theta h) = y_n + h sum_i w_i(theta) k_i,   theta in [0, 1],  theta1 = 1 - theta,
//   w_i(theta) = theta { b_i + theta1 [ (delta_i1 - b_i) + theta ( (2 b_i - delta_i1 - delta_i7) + theta1 d_i ) ] },
// b = the 5th-order weights (b_7 = 0), d = the dense-output coefficients below (d_2 = 0).  Properties pinned by
// tests/test_oracle_adaptive.py: w(0) = 0, w(1) = b, w'(0) = e_1, w'(1) = e_7 (a C^1 Hermite interpolant of the
// accepted steps) and the order conditions sum_i w_i(theta) Phi_i = theta^q / gamma for all trees up to q = 4.
template <class R> void dp45_dense_weights(R theta, R w[7]) {
    static const DP45 T;
    static const long double d[7] = {-12715105075.0L / 11282082432.0L, 0.0L, 87487479700.0L / 32700410799.0L,
                                     -10690763975.0L / 1880347072.0L, 701980252875.0L / 199316789632.0L,
                                     -1453857185.0L / 822651844.0L, 69997945.0L / 29380423.0L};
    const R th1 = R(1) - theta;
    for (int i = 0; i < 7; ++i) {
        const R b = (R)(i < 6 ? T.a[6][i] : 0.0L);
        const R e1 = i == 0 ? R(1) : R(0), e7 = i == 6 ? R(1) : R(0);
        w[i] = theta * (b + th1 * ((e1 - b) + theta * ((R(2) * b - e1 - e7) + th1 * (R)d[i])));
    }
}

}  // namespace
