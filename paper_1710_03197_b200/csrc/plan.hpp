// plan.hpp -- host-side (float64) planning of the NUFFT hot path: everything derived from the trajectory and the
// geometry is computed once, before any transform.
// Part of the product path; shares nothing with oracle/ (the Kaiser-Bessel functions below are this library's own
// float64 implementation: I0 by its power series, Phi by its closed form).
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>

#include "common.cuh"

namespace nufft {
namespace host {

constexpr double kPi = 3.14159265358979323846264338327950288;

// modified Bessel function of the first kind, order 0: sum_k (x^2/4)^k / (k!)^2
inline double bessel_i0(double x) {
    const double q = 0.25 * x * x;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

// Kaiser-Bessel shape parameter (reading R2): beta = pi sqrt((J/sigma)^2 (sigma - 1/2)^2 - 0.8)
inline double kb_beta(double J, double sigma) {
    return kPi * std::sqrt((J / sigma) * (J / sigma) * (sigma - 0.5) * (sigma - 0.5) - 0.8);
}

// phi(t) = I0(beta sqrt(1 - (2t/J)^2)) / I0(beta), |t| < J/2 (reading R1); the caller keeps |t| < J/2
inline double kb_phi(double t, double J, double beta) {
    double a = 1.0 - (2.0 * t / J) * (2.0 * t / J);
    if (a < 0.0) a = 0.0;
    return bessel_i0(beta * std::sqrt(a)) / bessel_i0(beta);
}

// Fourier transform of phi: Phi(xi) = J / I0(beta) * sinh(z)/z, z = sqrt(beta^2 - (pi J xi)^2)   (sin(z)/z beyond)
inline double kb_Phi(double xi, double J, double beta) {
    const double a = kPi * J * xi;
    const double z2 = beta * beta - a * a;
    double v;
    if (std::fabs(z2) < 1e-24) v = 1.0;
    else if (z2 > 0.0) { const double z = std::sqrt(z2); v = std::sinh(z) / z; }
    else { const double z = std::sqrt(-z2); v = std::sin(z) / z; }
    return J / bessel_i0(beta) * v;
}

// scaling factors s[n] = 1 / Phi((n - N/2)/K)   (reading R3), real, separable
inline std::vector<float> scaling_vector(int N, int K, double J) {
    const double beta = kb_beta(J, (double)K / (double)N);
    std::vector<float> s(N);
    for (int n = 0; n < N; ++n) s[n] = (float)(1.0 / kb_Phi(((double)n - 0.5 * N) / (double)K, J, beta));
    return s;
}

// twiddle table W_K^m = exp(-2 pi i m / K), m = 0..K-1, built in float64 and rounded once
inline std::vector<float2> twiddle_table(int K) {
    std::vector<float2> t(K);
    for (int m = 0; m < K; ++m) {
        const double a = -2.0 * kPi * (double)m / (double)K;
        t[m] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    return t;
}

// Degree-kPolyDeg polynomial interpolant (Chebyshev nodes, float64) of phi_j(z) = phi(J/2 - (z+1)/2 - j), z in
// [-1,1], j = 0 .. npieces-1, converted to the monomial basis and split into even / odd parts (see common.cuh
// KernelPoly / KernelPolyG).  Returns the max abs fit error over a fine mesh (over all pieces) in *max_err.
inline void fit_kernel_pieces(double J, double sigma, int npieces, float (*ev)[kPolyHalf], float (*od)[kPolyHalf],
                              double* max_err) {
    const double beta = kb_beta(J, sigma);
    constexpr int n = kPolyDeg + 1;
    double worst = 0.0;
    for (int j = 0; j < npieces; ++j) {
        auto f = [&](double z) { return kb_phi(0.5 * J - 0.5 * (z + 1.0) - (double)j, J, beta); };
        // Chebyshev coefficients from values at the n Chebyshev-Gauss nodes
        double fx[n], c[n];
        for (int i = 0; i < n; ++i) fx[i] = f(std::cos(kPi * (i + 0.5) / n));
        for (int k = 0; k < n; ++k) {
            double acc = 0.0;
            for (int i = 0; i < n; ++i) acc += fx[i] * std::cos(kPi * k * (i + 0.5) / n);
            c[k] = (k == 0 ? 1.0 : 2.0) * acc / n;
        }
        // sum_k c_k T_k(z) -> monomials, via T_{k+1} = 2 z T_k - T_{k-1}
        double mono[n] = {0}, Tkm1[n] = {0}, Tk[n] = {0}, Tn[n];
        Tkm1[0] = 1.0;           // T_0
        Tk[1] = 1.0;             // T_1
        mono[0] += c[0];
        if (n > 1) mono[1] += c[1];
        for (int k = 2; k < n; ++k) {
            for (int i = 0; i < n; ++i) Tn[i] = (i > 0 ? 2.0 * Tk[i - 1] : 0.0) - Tkm1[i];
            for (int i = 0; i < n; ++i) { mono[i] += c[k] * Tn[i]; Tkm1[i] = Tk[i]; Tk[i] = Tn[i]; }
        }
        for (int h = 0; h < kPolyHalf; ++h) { ev[j][h] = (float)mono[2 * h]; od[j][h] = (float)mono[2 * h + 1]; }
        for (int i = 0; i <= 2000; ++i) {
            const double z = -1.0 + i * 1e-3;
            double v = 0.0;
            for (int k = n - 1; k >= 0; --k) v = v * z + mono[k];
            const double e = std::fabs(v - f(z));
            if (e > worst) worst = e;
        }
    }
    if (max_err) *max_err = worst;
}
inline KernelPoly fit_kernel_poly(double J, double sigma, double* max_err) {      // J = kJ: three pairs
    KernelPoly P;
    fit_kernel_pieces(J, sigma, kJ / 2, P.ev, P.od, max_err);
    return P;
}
inline KernelPolyG fit_kernel_poly_g(int J, double sigma, double* max_err) {      // any J in [kJmin, kJmax]
    KernelPolyG P{};
    fit_kernel_pieces((double)J, sigma, (J + 1) / 2, P.ev, P.od, max_err);
    return P;
}

// Per-sample split of the coordinate, in float64 (reading R6/R11):
//   u = om * (K / (2 pi));  k0 = ceil(u - J/2);  delta = k0 - (u - J/2) in [0,1);  returns k0 mod K.
inline int split_coordinate(double om, int K, double J, float* delta, double* delta64 = nullptr) {
    const double u = om * ((double)K / (2.0 * kPi));
    const double k0 = std::ceil(u - 0.5 * J);
    double dl = k0 - (u - 0.5 * J);
    if (delta64) *delta64 = dl;
    float df = (float)dl;
    if (df >= 1.0f) df = 0.99999994f;      // float rounding of 1 - tiny; phi is continuous there
    *delta = df;
    long long k = (long long)k0 % K;
    if (k < 0) k += K;
    return (int)k;
}

// Six weights of one axis in float64: w[j] = phi(J/2 - delta - j), with phi(+J/2) = 0 (open support, reading R6).
inline void kb_weights_f64(double delta, double J, double beta, double (&w)[kJ]) {
    for (int j = 0; j < kJ; ++j) w[j] = kb_phi(0.5 * J - delta - (double)j, J, beta);
    if (delta == 0.0) w[0] = 0.0;
}

}  // namespace host
}  // namespace nufft
