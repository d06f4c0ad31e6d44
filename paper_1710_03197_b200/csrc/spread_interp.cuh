// spread_interp.cuh -- V (interpolation, step a3) and V^H (gridding, step a4) of the NUFFT hot path.
// V is the M x prod(Kd) sparse interpolation matrix with prod(Jd) non-zeros per row, V^H its
// conjugate transpose.  The paper stores V (and a second copy for V^H) as CSR with complex64 values; here no matrix
// is stored: each sample carries a packed base index and d fractions (4 + 4d bytes) and the prod(Jd) real weights
// are recomputed on the fly from the separable Kaiser-Bessel kernel (common.cuh, kb_weights).
#pragma once
#include "common.cuh"

namespace nufft {

struct GridGeom {
    int K[3];              // grid size per axis (K[2] = 1 when d == 2 is NOT used; see D template parameter)
    int64_t cells;         // prod K  (= batch stride of a [batch][grid] array)
    int64_t M;             // samples (= batch stride of y)
};

// Per-sample plan data, in TILE-SORTED order (position i of the sorted order is caller sample perm[i]).
struct SampleData {
    const uint32_t* kpack; // base index k0 mod K of the stencil per axis, 10 bits each (axis 0 in bits 0..9)
    const float* delta;    // [d][M]: delta_a = k0_a - (u_a - J/2) in [0,1)
    const int32_t* perm;   // sorted position -> caller's sample index
};

__device__ __forceinline__ void unpack_k0(uint32_t kp, int (&k0)[3]) {
    k0[0] = kp & 1023u; k0[1] = (kp >> 10) & 1023u; k0[2] = (kp >> 20) & 1023u;
}

// ------------------------------------------------------------------------------------------------------------
// V, direct form: one thread per sample (tile-sorted order, so a warp's stencils share cache lines), the prod(J)
// stencil values gathered straight from the grid through L1/L2.  y is written in the caller's order.
// ------------------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128)
interp_direct_kernel(SampleData s, GridGeom g, const float2* __restrict__ grid, float2* __restrict__ y, KernelPoly P) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.M) return;
    const int b = blockIdx.y;
    int k0[3];
    unpack_k0(__ldg(&s.kpack[i]), k0);
    float w[D][kJ];
#pragma unroll
    for (int a = 0; a < D; ++a) kb_weights(P, __ldg(&s.delta[(int64_t)a * g.M + i]), w[a]);
    const float2* __restrict__ G = grid + (int64_t)b * g.cells;
    float2 acc = make_float2(0.f, 0.f);
    if (D == 2) {
        const int K0 = g.K[0], K1 = g.K[1];
#pragma unroll
        for (int j0 = 0; j0 < kJ; ++j0) {
            const float2* __restrict__ row = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1;
            float2 r = make_float2(0.f, 0.f);
#pragma unroll
            for (int j1 = 0; j1 < kJ; ++j1) {
                const float2 v = __ldg(&row[(k0[1] + j1) & (K1 - 1)]);
                r.x = fmaf(w[1][j1], v.x, r.x);
                r.y = fmaf(w[1][j1], v.y, r.y);
            }
            acc.x = fmaf(w[0][j0], r.x, acc.x);
            acc.y = fmaf(w[0][j0], r.y, acc.y);
        }
    } else {
        const int K0 = g.K[0], K1 = g.K[1], K2 = g.K[2];
#pragma unroll 1
        for (int j0 = 0; j0 < kJ; ++j0) {
            const float2* __restrict__ plane = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1 * K2;
            float2 rp = make_float2(0.f, 0.f);
#pragma unroll
            for (int j1 = 0; j1 < kJ; ++j1) {
                const float2* __restrict__ row = plane + (int64_t)((k0[1] + j1) & (K1 - 1)) * K2;
                float2 r = make_float2(0.f, 0.f);
#pragma unroll
                for (int j2 = 0; j2 < kJ; ++j2) {
                    const float2 v = __ldg(&row[(k0[2] + j2) & (K2 - 1)]);
                    r.x = fmaf(w[D - 1][j2], v.x, r.x);
                    r.y = fmaf(w[D - 1][j2], v.y, r.y);
                }
                rp.x = fmaf(w[1][j1], r.x, rp.x);
                rp.y = fmaf(w[1][j1], r.y, rp.y);
            }
            const float w0 = w[0][j0];
            acc.x = fmaf(w0, rp.x, acc.x);
            acc.y = fmaf(w0, rp.y, acc.y);
        }
    }
    y[(int64_t)b * g.M + __ldg(&s.perm[i])] = acc;
}

// ------------------------------------------------------------------------------------------------------------
// V^H, baseline form: one thread per sample, one vector atomic (red.global.add.v2.f32) per stencil point into a
// zeroed grid.  Kept as the simple fallback / cross-check of the tiled kernels.
// ------------------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128)
gridding_atomic_kernel(SampleData s, GridGeom g, const float2* __restrict__ y, float2* __restrict__ grid, KernelPoly P) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.M) return;
    const int b = blockIdx.y;
    int k0[3];
    unpack_k0(__ldg(&s.kpack[i]), k0);
    float w[D][kJ];
#pragma unroll
    for (int a = 0; a < D; ++a) kb_weights(P, __ldg(&s.delta[(int64_t)a * g.M + i]), w[a]);
    const float2 yv = __ldg(&y[(int64_t)b * g.M + __ldg(&s.perm[i])]);
    float2* __restrict__ G = grid + (int64_t)b * g.cells;
    if (D == 2) {
        const int K0 = g.K[0], K1 = g.K[1];
#pragma unroll
        for (int j0 = 0; j0 < kJ; ++j0) {
            float2* __restrict__ row = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1;
            const float2 yr = cscale(yv, w[0][j0]);
#pragma unroll
            for (int j1 = 0; j1 < kJ; ++j1) atomicAdd(&row[(k0[1] + j1) & (K1 - 1)], cscale(yr, w[1][j1]));
        }
    } else {
        const int K0 = g.K[0], K1 = g.K[1], K2 = g.K[2];
#pragma unroll 1
        for (int j0 = 0; j0 < kJ; ++j0) {
            float2* __restrict__ plane = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1 * K2;
            const float2 yp = cscale(yv, w[0][j0]);
#pragma unroll
            for (int j1 = 0; j1 < kJ; ++j1) {
                float2* __restrict__ row = plane + (int64_t)((k0[1] + j1) & (K1 - 1)) * K2;
                const float2 yr = cscale(yp, w[1][j1]);
#pragma unroll
                for (int j2 = 0; j2 < kJ; ++j2) atomicAdd(&row[(k0[2] + j2) & (K2 - 1)], cscale(yr, w[D - 1][j2]));
            }
        }
    }
}

}  // namespace nufft
