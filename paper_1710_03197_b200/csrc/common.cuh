// common.cuh -- small shared helpers of the CUDA path (complex arithmetic, error plumbing).
// Part of the product path; shares nothing with oracle/.
#pragma once
#include <cuda.h>
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

constexpr int kJ = 6;          // interpolation kernel width in grid cells (Jd) of the tuned (tiled / interleaved) kernels
constexpr int kJmin = 2;       // other widths kJmin..kJmax run on the direct V / atomic V^H kernels
constexpr int kJmax = 8;
constexpr int kPolyDeg = 9;    // degree of the piecewise polynomial fit of the Kaiser-Bessel kernel
constexpr int kPolyHalf = 5;   // even / odd coefficient count ((kPolyDeg + 1) / 2)

// Piecewise polynomial fit of phi(J/2 - delta - j), j = 0..5, delta in [0,1), in z = 2 delta - 1.
// By symmetry phi_{5-j}(z) = phi_j(-z), so three even/odd pairs describe all six pieces:
//   phi_j(z) = ev[j](z^2) + z od[j](z^2),   phi_{5-j}(z) = ev[j](z^2) - z od[j](z^2),   j = 0,1,2.
// One set per grid axis: the kernel shape depends on the axis through sigma_a = K_a / N_a (beta, reading R2) and, for the
// min-max interpolator, through N_a itself (reading R25).
struct KernelPoly {
    float ev[3][3][kPolyHalf];      // [axis][piece][coefficient]
    float od[3][3][kPolyHalf];
    float zero_at;     // delta at which w[0] is exactly zero: 0 for Kaiser-Bessel (open support, R6), -1 (never) for min-max
};

// Six interpolation weights of one axis: w[j] = phi(J/2 - delta - j).
// delta == 0 means the sample sits on a grid point: phi(+J/2) = 0 exactly (open support, reading R6).
__device__ __forceinline__ void kb_weights(const KernelPoly& P, int a, float delta, float (&w)[kJ]) {
    const float z = fmaf(2.0f, delta, -1.0f);
    const float z2 = z * z;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        float e = P.ev[a][j][kPolyHalf - 1], o = P.od[a][j][kPolyHalf - 1];
#pragma unroll
        for (int c = kPolyHalf - 2; c >= 0; --c) {
            e = fmaf(e, z2, P.ev[a][j][c]);
            o = fmaf(o, z2, P.od[a][j][c]);
        }
        o *= z;
        w[j] = e + o;
        w[kJ - 1 - j] = e - o;
    }
    if (delta == P.zero_at) w[0] = 0.0f;
}

// Any width J in [kJmin, kJmax]: ceil(J/2) even/odd pairs, phi_{J-1-j}(z) = phi_j(-z) (for odd J the middle piece is its
// own mirror image).  With J = 6 and KernelPoly this is kb_weights above.
struct KernelPolyG {
    float ev[3][(kJmax + 1) / 2][kPolyHalf];
    float od[3][(kJmax + 1) / 2][kPolyHalf];
    float zero_at;
};

template <int J, class Poly>
__device__ __forceinline__ void kb_weights_j(const Poly& P, int a, float delta, float (&w)[J]) {
    const float z = fmaf(2.0f, delta, -1.0f);
    const float z2 = z * z;
#pragma unroll
    for (int j = 0; j < (J + 1) / 2; ++j) {
        float e = P.ev[a][j][kPolyHalf - 1], o = P.od[a][j][kPolyHalf - 1];
#pragma unroll
        for (int c = kPolyHalf - 2; c >= 0; --c) {
            e = fmaf(e, z2, P.ev[a][j][c]);
            o = fmaf(o, z2, P.od[a][j][c]);
        }
        o *= z;
        w[j] = e + o;
        if (J - 1 - j != j) w[J - 1 - j] = e - o;
    }
    if (delta == P.zero_at) w[0] = 0.0f;
}

#ifdef __CUDACC__
// ---- bulk-copy staging helpers (cp.async.bulk + mbarrier: the TMA engine moves contiguous plan / sample ranges into
// shared memory; SASS: UBLKCP, SYNCS) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// shared -> global bulk REDUCTION (element-wise f32 add performed by the TMA engine at L2): used to flush accumulated tiles
__device__ __forceinline__ void bulk_s2g_add_f32(void* gdst, const void* ssrc, uint32_t bytes) {
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;"
                 ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit_and_wait_read() {
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// ---- tensor-map TMA (cp.async.bulk.tensor, SASS UTMALDG / UTMAREDG): ONE copy moves the whole padded tile
// (24 x 13 x 13 cells) between the grid and shared memory.  round 2: with one 192-byte cp.async.bulk per padded row
// (169 per CTA, 1.9 M per launch) the per-SM TMA issue rate, not bandwidth, bounded both 3-D kernels at ~0.24 ms.
// The map views the planar grid [B][K0][K1][K2] complex64 as float32 [B][K0][K1][2 K2]; box = {48, 13, 13, 1}.  Tiles
// whose padded box crosses the periodic seam keep the row-copy path (a tensor box cannot wrap).
__device__ __forceinline__ void tma_load_tile_4d(void* smem_dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3,
                                                 uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(smem_dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_reduce_add_tile_4d(const CUtensorMap* tm, int c0, int c1, int c2, int c3,
                                                       const void* smem_src) {
    asm volatile("cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                 ::"l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(smem_src)) : "memory");
}

// 2-D planar grid [B][K0][K1] complex64 seen as float32 [B][K0][2 K1]; box = {2 pitch, P0, 1}
__device__ __forceinline__ void tma_load_tile_3d(void* smem_dst, const CUtensorMap* tm, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(smem_dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_reduce_add_tile_3d(const CUtensorMap* tm, int c0, int c1, int c2, const void* smem_src) {
    asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2, %3}], [%4];"
                 ::"l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(smem_src)) : "memory");
}

// Programmatic dependent launch (PDL): a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start
// while its predecessor in the stream is still running; pdl_enter() is its first statement: it lets the NEXT kernel in the
// stream be scheduled early (launch_dependents) and then waits until the predecessor grid has completed and its writes are
// visible (wait).  Without the launch attribute both are no-ops.  The small dependent kernels of a single transform then
// overlap their launch latency and CTA scheduling with the tail of the previous kernel.
__device__ __forceinline__ void pdl_enter() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}

#endif

}  // namespace nufft
