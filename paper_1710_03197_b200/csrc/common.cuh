// common.cuh -- small shared helpers of the CUDA path (complex arithmetic, error plumbing).
// Part of the product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nufft {

__host__ __device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__host__ __device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__host__ __device__ __forceinline__ float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
__host__ __device__ __forceinline__ float2 cscale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }
// a * (-i)
__host__ __device__ __forceinline__ float2 cmul_mi(float2 a) { return make_float2(a.y, -a.x); }

constexpr int kJ = 6;          // interpolation kernel width in grid cells (Jd), the one supported value
constexpr int kPolyDeg = 9;    // degree of the piecewise polynomial fit of the Kaiser-Bessel kernel
constexpr int kPolyHalf = 5;   // even / odd coefficient count ((kPolyDeg + 1) / 2)

// Piecewise polynomial fit of phi(J/2 - delta - j), j = 0..5, delta in [0,1), in z = 2 delta - 1.
// By symmetry phi_{5-j}(z) = phi_j(-z), so three even/odd pairs describe all six pieces:
//   phi_j(z) = ev[j](z^2) + z od[j](z^2),   phi_{5-j}(z) = ev[j](z^2) - z od[j](z^2),   j = 0,1,2.
struct KernelPoly {
    float ev[3][kPolyHalf];
    float od[3][kPolyHalf];
};

// Six interpolation weights of one axis: w[j] = phi(J/2 - delta - j).
// delta == 0 means the sample sits on a grid point: phi(+J/2) = 0 exactly (open support, reading R6).
__device__ __forceinline__ void kb_weights(const KernelPoly& P, float delta, float (&w)[kJ]) {
    const float z = fmaf(2.0f, delta, -1.0f);
    const float z2 = z * z;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        float e = P.ev[j][kPolyHalf - 1], o = P.od[j][kPolyHalf - 1];
#pragma unroll
        for (int c = kPolyHalf - 2; c >= 0; --c) {
            e = fmaf(e, z2, P.ev[j][c]);
            o = fmaf(o, z2, P.od[j][c]);
        }
        o *= z;
        w[j] = e + o;
        w[kJ - 1 - j] = e - o;
    }
    if (delta == 0.0f) w[0] = 0.0f;
}

}  // namespace nufft
