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

// Degree-kPolyDeg polynomial interpolant (Chebyshev nodes, float64) of the kernel pieces f(j, z), z in [-1,1]
// (z = 2 delta - 1), j = 0 .. npieces-1, converted to the monomial basis and split into even / odd parts (see common.cuh
// KernelPoly / KernelPolyG).  Returns the max abs fit error over a fine mesh (over all pieces) in *max_err.
template <class F>
inline void fit_pieces(F f, int npieces, float (*ev)[kPolyHalf], float (*od)[kPolyHalf], double* max_err) {
    constexpr int n = kPolyDeg + 1;
    double worst = 0.0;
    for (int j = 0; j < npieces; ++j) {
        // Chebyshev coefficients from values at the n Chebyshev-Gauss nodes
        double fx[n], c[n];
        for (int i = 0; i < n; ++i) fx[i] = f(j, std::cos(kPi * (i + 0.5) / n));
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
            const double e = std::fabs(v - f(j, z));
            if (e > worst) worst = e;
        }
    }
    if (max_err) *max_err = worst;
}

// Kaiser-Bessel pieces: phi_j(z) = phi(J/2 - (z+1)/2 - j)
inline void fit_kernel_pieces(double J, double sigma, int npieces, float (*ev)[kPolyHalf], float (*od)[kPolyHalf],
                              double* max_err) {
    const double beta = kb_beta(J, sigma);
    fit_pieces([&](int j, double z) { return kb_phi(0.5 * J - 0.5 * (z + 1.0) - (double)j, J, beta); }, npieces, ev, od,
               max_err);
}
// one axis of a KernelPoly / KernelPolyG: pieces = ceil(J/2)
template <class Poly>
inline void fit_kernel_axis(Poly& P, int a, int J, double sigma, double* max_err) {
    fit_kernel_pieces((double)J, sigma, (J + 1) / 2, P.ev[a], P.od[a], max_err);
}

// ------------------------------------------------------------------------------------------------------------
// Min-max interpolator with Kaiser-Bessel scaling factors ("the default kernel is the min-max kernel";
// SURVEY 8(f)-4; reading R25): for stencil offsets t_l = J/2 - delta - l the J real weights solve
//     T w = r(delta),   T[l][j] = sum_p c_p s_p^2 cos(gamma (l - j) p),   r[l] = sum_p c_p s_p cos(gamma t_l p),
// p = -N/2 .. N/2 with c = 1/2 at both ends (= the image's own N pixels, the summands being even), s_p = 1 / Phi(p / K).
// The weights are analytic in delta: they are sampled once per plan at 32 Chebyshev nodes (32 solves) and every later
// evaluation -- the float64 V^H table and the fit of the device polynomial -- goes through that interpolant.
// ------------------------------------------------------------------------------------------------------------
struct MinMaxKernel {
    static constexpr int kNodes = 32;
    int J = 0;
    double cheb[kJmax][kNodes];      // Chebyshev coefficients of w_j(z), z = 2 delta - 1

    void build(int N, int K, int Jw) {
        J = Jw;
        const double beta = kb_beta((double)J, (double)K / (double)N), gam = 2.0 * kPi / (double)K;
        const int np = N + 1;
        std::vector<double> pp(np), cs(np), css(np);
        for (int i = 0; i < np; ++i) {
            pp[i] = (double)(i - N / 2);
            const double sv = 1.0 / kb_Phi(pp[i] / (double)K, (double)J, beta);
            const double c = (i == 0 || i == np - 1) ? 0.5 : 1.0;
            cs[i] = c * sv;
            css[i] = c * sv * sv;
        }
        double T[kJmax][kJmax];
        for (int l = 0; l < J; ++l)
            for (int j = 0; j < J; ++j) {
                double acc = 0.0;
                for (int i = 0; i < np; ++i) acc += css[i] * std::cos(gam * (double)(l - j) * pp[i]);
                T[l][j] = acc;
            }
        double wn[kNodes][kJmax];
        for (int q = 0; q < kNodes; ++q) {
            const double z = std::cos(kPi * (q + 0.5) / kNodes), delta = 0.5 * (z + 1.0);
            double A[kJmax][kJmax + 1];
            for (int l = 0; l < J; ++l) {
                const double t = 0.5 * J - delta - (double)l;
                double acc = 0.0;
                for (int i = 0; i < np; ++i) acc += cs[i] * std::cos(gam * t * pp[i]);
                for (int j = 0; j < J; ++j) A[l][j] = T[l][j];
                A[l][J] = acc;
            }
            // Gaussian elimination with partial pivoting (T is symmetric positive definite, cond <= 1e5 for J <= 8)
            for (int c = 0; c < J; ++c) {
                int piv = c;
                for (int r2 = c + 1; r2 < J; ++r2) if (std::fabs(A[r2][c]) > std::fabs(A[piv][c])) piv = r2;
                if (piv != c) for (int k = 0; k <= J; ++k) std::swap(A[c][k], A[piv][k]);
                for (int r2 = c + 1; r2 < J; ++r2) {
                    const double f = A[r2][c] / A[c][c];
                    for (int k = c; k <= J; ++k) A[r2][k] -= f * A[c][k];
                }
            }
            for (int r2 = J - 1; r2 >= 0; --r2) {
                double acc = A[r2][J];
                for (int k = r2 + 1; k < J; ++k) acc -= A[r2][k] * wn[q][k];
                wn[q][r2] = acc / A[r2][r2];
            }
        }
        for (int j = 0; j < J; ++j)
            for (int k = 0; k < kNodes; ++k) {
                double acc = 0.0;
                for (int q = 0; q < kNodes; ++q) acc += wn[q][j] * std::cos(kPi * k * (q + 0.5) / kNodes);
                cheb[j][k] = (k == 0 ? 1.0 : 2.0) * acc / kNodes;
            }
    }
    // w_j at z = 2 delta - 1 (Clenshaw)
    double eval(int j, double z) const {
        double b1 = 0.0, b2 = 0.0;
        for (int k = kNodes - 1; k >= 1; --k) { const double b0 = 2.0 * z * b1 - b2 + cheb[j][k]; b2 = b1; b1 = b0; }
        return z * b1 - b2 + cheb[j][0];
    }
    void weights(double delta, double* w) const {
        const double z = 2.0 * delta - 1.0;
        for (int j = 0; j < J; ++j) w[j] = eval(j, z);
    }
    template <class Poly> void fit_axis(Poly& P, int a, double* max_err) const {
        fit_pieces([&](int j, double z) { return eval(j, z); }, (J + 1) / 2, P.ev[a], P.od[a], max_err);
        P.zero_at = -1.0f;        // no open-support zero: the weight at t = J/2 is whatever the least-squares solution gives
    }
};

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
