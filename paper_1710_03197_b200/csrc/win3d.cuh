// win3d.cuh -- register-window V (step a3) and V^H (step a4) for 3-D plans at Jd = 6.
//
// Why.  profiles/r01i: the tile-staged 3-D kernels of round 1 are bound by the shared-memory data pipe, not by HBM:
// every sample re-reads (V) or read-modify-writes (V^H) its whole 6 x 6 x 6 stencil in shared memory, 27.7 / 49
// wavefronts per sample.  A kooshball readout advances half a grid cell per sample, so neighbouring samples share
// almost all of their stencil; here that overlap is kept in REGISTERS:
//
//   * a work item is (tile 8 x 8 x 16 cells, range of tile-sorted samples) as before, and the padded tile
//     (13 x 13 x 24 cells) lives in shared memory (V: staged by cp.async.bulk; V^H: zeroed, flushed by
//     cp.reduce.async.bulk);
//   * inside a tile the plan sorts the samples by PENCIL -- a 3 x 3 block of stencil base cells on axes 0, 1 -- and then
//     by base cell on axis 2.  All stencils of a pencil lie inside an 8 x 8 window on axes 0, 1;
//   * every warp walks a contiguous share of the item's samples and holds a WINDOW of 8 planes x 8 rows x 8 columns of
//     grid cells in registers: lane (y, q) owns row y and ONE pair of adjacent columns (a 16-byte float4) in each of the
//     8 planes = 32 registers.  The window slides along axis 2 with the sorted samples: when the base pair advances,
//     only the lanes whose pair leaves the window flush it (V^H: one float4 read-modify-write per plane under the
//     tile's lock) or load the pair that enters (V);
//   * a sample costs five small shared-memory loads (its zero-padded weight vectors, written once per sample by the
//     lane that evaluated the kernel polynomial) and 16 packed FMAs (FFMA2) per lane; V sums the 32 partial results
//     of eight samples at a time with a transposing shuffle reduction (18 shuffles per 8 samples instead of 80).
//
// The weights outside a sample's 6-cell support are exact zeros, so the arithmetic is that of the plain stencil sum.
#pragma once
#include "common.cuh"
#include "spread_interp.cuh"

namespace nufft {

constexpr int kW3Rec = 28;                  // floats per staged sample record (7 float4; 7 s mod 8 is a permutation:
                                            // the 128-bit stores of 8 consecutive lanes fall into distinct bank quads)
// warps per CTA of the register-window 3-D kernels (win3d.cuh), measured on config 4 (profiles/r02_cfg4_3d.md):
// V 1 / 2 / 4 / 8 warps: 0.304 / 0.249 / 0.217 / 0.258 ms;  V^H (1 warp = no tile lock): 0.315 / 0.386 / 0.491 / 0.927 ms
constexpr int kW3InterpWarps = 4, kW3GridWarps = 1;
// NW warps per CTA: tile + NW x 32 records + mbarrier / lock
constexpr int win3d_smem(int nw) { return k3Cells * 8 + nw * 32 * kW3Rec * 4 + 16 + nw * 16; }   // + 2 mbarriers per warp (TABLE)

// tile-local stencil base (c0, c1, c2) -> window: pencil base on axes 0, 1 (blocks of 3 cells, the last block of the
// 8-cell tile edge holds 2), base PAIR on axis 2
__host__ __device__ __forceinline__ int w3_block_base(int c) { return c >= 6 ? 5 : (c / 3) * 3; }
// sort key of a sample inside its tile (plan time): pencil, then base pair on axis 2
__host__ __device__ __forceinline__ int w3_sub_key(int c0, int c1, int c2) {
    return ((c0 >= 6 ? 2 : c0 / 3) * 3 + (c1 >= 6 ? 2 : c1 / 3)) * 8 + (c2 >> 1);
}
constexpr int kW3SubKeys = 9 * 8;

// zero-padded weight vector: p[i] = w[i - o], 0 <= i - o < 6, else 0   (o in {0, 1, 2})
__device__ __forceinline__ void w3_pad(const float (&w)[kJ], int o, float4& a, float4& b) {
    const bool o0 = o == 0, o1 = o == 1;
    a.x = o0 ? w[0] : 0.f;
    a.y = o0 ? w[1] : (o1 ? w[0] : 0.f);
    a.z = o0 ? w[2] : (o1 ? w[1] : w[0]);
    a.w = o0 ? w[3] : (o1 ? w[2] : w[1]);
    b.x = o0 ? w[4] : (o1 ? w[3] : w[2]);
    b.y = o0 ? w[5] : (o1 ? w[4] : w[3]);
    b.z = o0 ? 0.f : (o1 ? w[5] : w[4]);
    b.w = (o0 || o1) ? 0.f : w[5];
}

// Plan data of one sample, fetched one chunk ahead of its use (the global-load latency hides behind the previous chunk)
struct W3Pre {
    uint32_t kp;
    float d0, d1, d2;
    int m;            // caller's sample index, -1 = no sample
    float2 yv;        // V^H only
};
__device__ __forceinline__ void w3_fetch(const SampleData& s, const GridGeom& g, int si, bool valid, W3Pre& f) {
    f.m = -1; f.kp = 0; f.d0 = f.d1 = f.d2 = 0.f; f.yv = make_float2(0.f, 0.f);
    if (valid) {
        f.kp = __ldg(&s.kpack[si]);
        f.d0 = __ldg(&s.delta[si]);
        f.d1 = __ldg(&s.delta[g.M + si]);
        f.d2 = __ldg(&s.delta[2 * g.M + si]);
        f.m = __ldg(&s.perm[si]);
    }
}
// One lane prepares the record of one sample of the item:
//   [0..7] w0 padded, [8..15] w1 padded, [16..23] w2 padded relative to the base pair and rotated by it, [24] window key
//   ((tile cell offset of the pencil base) << 4 | base pair), [25] caller's sample index, [26..27] y (V^H)
__device__ __forceinline__ void w3_stage(const W3Pre& f, const GridGeom& g, const KernelPoly& P, const int (&o)[3], float* rec) {
    float4 r0, r1, r2, r3, r4, r5, r6;
    if (f.m >= 0) {
        int k0[3];
        unpack_k0(f.kp, k0);
        const int c0 = (k0[0] - o[0]) & (g.K[0] - 1), c1 = (k0[1] - o[1]) & (g.K[1] - 1), c2 = (k0[2] - o[2]) & (g.K[2] - 1);
        const int b0 = w3_block_base(c0), b1 = w3_block_base(c1), zb = c2 >> 1;
        float w[kJ];
        kb_weights(P, 0, f.d0, w);
        w3_pad(w, c0 - b0, r0, r1);
        kb_weights(P, 1, f.d1, w);
        w3_pad(w, c1 - b1, r2, r3);
        kb_weights(P, 2, f.d2, w);
        {   // axis 2: padded relative to the base pair, then ROTATED by the base pair: slot ((zb + i) & 3) holds pair i of
            // the window, so that lane (y, q), which owns the pair = q (mod 4), always reads slot q
            float4 a, b;
            w3_pad(w, c2 & 1, a, b);
            const int rot = zb & 3;
            const float2 P0 = make_float2(a.x, a.y), P1 = make_float2(a.z, a.w), P2 = make_float2(b.x, b.y), P3 = make_float2(b.z, b.w);
            const float2 R0 = rot == 0 ? P0 : (rot == 1 ? P3 : (rot == 2 ? P2 : P1));
            const float2 R1 = rot == 0 ? P1 : (rot == 1 ? P0 : (rot == 2 ? P3 : P2));
            const float2 R2 = rot == 0 ? P2 : (rot == 1 ? P1 : (rot == 2 ? P0 : P3));
            const float2 R3 = rot == 0 ? P3 : (rot == 1 ? P2 : (rot == 2 ? P1 : P0));
            r4 = make_float4(R0.x, R0.y, R1.x, R1.y);
            r5 = make_float4(R2.x, R2.y, R3.x, R3.y);
        }
        const int key = ((b0 * k3Plane + b1 * k3Pitch) << 4) | zb;
        r6 = make_float4(__int_as_float(key), __int_as_float(f.m), f.yv.x, f.yv.y);
    } else {        // past the end of the range: zero weights, nothing is written (the walk keeps its window)
        r0 = r1 = r2 = r3 = r4 = r5 = make_float4(0.f, 0.f, 0.f, 0.f);
        r6 = make_float4(__int_as_float(0), __int_as_float(-1), 0.f, 0.f);
    }
    float4* r = reinterpret_cast<float4*>(rec);
    r[0] = r0; r[1] = r1; r[2] = r2; r[3] = r3; r[4] = r4; r[5] = r5; r[6] = r6;
}

// share of warp `warp` of an item of n samples, in units of 8 samples (the V kernel reduces 8 samples at a time)
template <int NW>
__device__ __forceinline__ void w3_share(const WorkItem& wi, int warp, int& wb, int& we) {
    const int n = wi.s_end - wi.s_begin, u = (n + 7) >> 3;
    wb = min(wi.s_end, wi.s_begin + 8 * ((u * warp) / NW));
    we = min(wi.s_end, wi.s_begin + 8 * ((u * (warp + 1)) / NW));
}

__device__ __forceinline__ float2 w3_dup(float w) { return make_float2(w, w); }

// What lane (y, q) reads of a staged record: every address is lane-constant, so the loads of sample i + 1 are issued before
// sample i is applied (software pipeline; the walk is otherwise a chain of shared-memory load latencies)
struct W3Rec {
    float4 wa, wb;     // w0 padded (uniform)
    float w1;          // w1 padded [y]
    float2 w2;         // w2 of this lane's pair
    float4 kk;         // key, caller's sample index, y.re, y.im
};
__device__ __forceinline__ W3Rec w3_load(const float* r, int ly, int q) {
    W3Rec c;
    c.wa = *reinterpret_cast<const float4*>(r);
    c.wb = *reinterpret_cast<const float4*>(r + 4);
    c.w1 = r[8 + ly];
    c.w2 = *reinterpret_cast<const float2*>(r + 16 + 2 * q);
    c.kk = *reinterpret_cast<const float4*>(r + 24);
    return c;
}

// ------------------------------------------------------------------------------------------------------------
// V: y[m] = sum over the window of w0 w1 w2 G
// ------------------------------------------------------------------------------------------------------------
// TABLE (opts.coef_mode = 1): the sample records come precomputed from the plan (w3rec, 112 B per sample in walk order)
// and are moved into shared memory by one bulk copy per 16 samples, double-buffered per warp, instead of being evaluated
// from the kernel polynomial by one lane per sample.
template <int NW, bool TABLE>
__global__ void __launch_bounds__(NW * 32)
interp_win_3d_kernel(SampleData s, GridGeom g, const WorkItem* __restrict__ items, const float2* __restrict__ grid,
                     float2* __restrict__ y, KernelPoly P, const __grid_constant__ CUtensorMap tmap, int use_tmap,
                     const float* __restrict__ w3rec) {
    constexpr int CH = TABLE ? 16 : 32;
    extern __shared__ __align__(1024) unsigned char w3smem[];
    float2* tile = reinterpret_cast<float2*>(w3smem);
    float* recs = reinterpret_cast<float*>(tile + k3Cells);
    uint64_t* bar = reinterpret_cast<uint64_t*>(recs + NW * 32 * kW3Rec);
    const WorkItem wi = items[blockIdx.x];
    const int b = blockIdx.y;
    int o[3];
    unpack_k0(wi.origin, o);
    const int K0 = g.K[0], K1 = g.K[1], K2 = g.K[2];
    const float2* __restrict__ G = grid + (int64_t)b * g.cells;
    // stage the padded tile: one bulk copy per 24-cell row (rows wrap periodically, a row crossing the seam of the last
    // axis is split)
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_expect_tx(bar, (uint32_t)(k3P0 * k3P1 * k3Pitch * 8));
    }
    __syncthreads();
    const bool boxed = use_tmap && o[0] + k3P0 <= K0 && o[1] + k3P1 <= K1 && o[2] + k3Pitch <= K2;
    if (boxed) {
        if (threadIdx.x == 0) tma_load_tile_4d(tile, &tmap, 2 * o[2], o[1], o[0], b, bar);
    } else {
        for (int row = threadIdx.x; row < k3P0 * k3P1; row += blockDim.x) {
            const int lx = row / k3P1, ly = row - lx * k3P1;
            const int gx = (o[0] + lx) & (K0 - 1), gy = (o[1] + ly) & (K1 - 1), gz = o[2] & (K2 - 1);
            const float2* src = G + ((int64_t)gx * K1 + gy) * K2;
            float2* dst = tile + row * k3Pitch;
            const int first = min(k3Pitch, K2 - gz);
            bulk_g2s(dst, src + gz, (uint32_t)first * 8, bar);
            if (first < k3Pitch) bulk_g2s(dst + first, src, (uint32_t)(k3Pitch - first) * 8, bar);
        }
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ly = lane >> 2, q = lane & 3;
    float* rec = recs + warp * 32 * kW3Rec;
    float2* __restrict__ yb = y + (int64_t)b * g.M;
    // this warp's share of the item's samples
    int wb, we;
    w3_share<NW>(wi, warp, wb, we);
    float2 win[8][2];
#pragma unroll
    for (int p = 0; p < 8; ++p) { win[p][0] = make_float2(0.f, 0.f); win[p][1] = make_float2(0.f, 0.f); }
    int cur = -1;
    bool tile_ready = false;
    W3Pre pre;
    uint64_t* wbar = reinterpret_cast<uint64_t*>(reinterpret_cast<unsigned char*>(bar) + 16) + 2 * warp;
    float* const rec0 = rec;
    if (TABLE) {
        if (lane == 0) {
            mbar_init(&wbar[0], 1);
            mbar_init(&wbar[1], 1);
            if (wb < we) {
                const int n0 = min(CH, we - wb);
                mbar_expect_tx(&wbar[0], (uint32_t)n0 * kW3Rec * 4);
                bulk_g2s(rec0, w3rec + (int64_t)wb * kW3Rec, (uint32_t)n0 * kW3Rec * 4, &wbar[0]);
            }
        }
        __syncwarp();
    } else {
        w3_fetch(s, g, wb + lane, wb + lane < we, pre);
    }
    int it = 0;
    for (int c0 = wb; c0 < we; c0 += CH, ++it) {
        const int cnt = min(CH, we - c0);
        if (TABLE) {
            rec = rec0 + (it & 1) * CH * kW3Rec;
            if (lane == 0 && c0 + CH < we) {      // the other buffer was consumed one iteration ago (syncwarp at its end)
                const int n1 = min(CH, we - c0 - CH);
                mbar_expect_tx(&wbar[(it + 1) & 1], (uint32_t)n1 * kW3Rec * 4);
                bulk_g2s(rec0 + ((it + 1) & 1) * CH * kW3Rec, w3rec + (int64_t)(c0 + CH) * kW3Rec, (uint32_t)n1 * kW3Rec * 4,
                         &wbar[(it + 1) & 1]);
            }
            mbar_wait(&wbar[it & 1], (uint32_t)((it >> 1) & 1));
        } else {
            w3_stage(pre, g, P, o, rec + lane * kW3Rec);
            w3_fetch(s, g, c0 + 32 + lane, c0 + 32 + lane < we, pre);      // next chunk's plan data: in flight during this chunk
        }
        __syncwarp();
        if (!tile_ready) { mbar_wait(bar, 0); tile_ready = true; }
        W3Rec nx = w3_load(rec, ly, q);
#pragma unroll 1
        for (int s8 = 0; s8 < cnt; s8 += 8) {
            float2 part[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const W3Rec c = nx;
                nx = w3_load(rec + min(s8 + j + 1, CH - 1) * kW3Rec, ly, q);
                const int key = __float_as_int(c.kk.x);
                if (s8 + j < cnt && key != cur) {       // (slots past the end of a short chunk keep the window)
                    // slide (same pencil, base pair advanced by 1..3) or reload: lane (y, q) owns pair zb + ((q - zb) & 3)
                    const int zb = key & 15;
                    const bool same = cur >= 0 && (key >> 4) == (cur >> 4);
                    const int steps = same ? zb - (cur & 15) : 4;
                    const int zc = cur & 15;
                    const bool mine = (steps < 0 || steps >= 4) || (((q - zc) & 3) < steps);
                    if (mine) {
                        const float2* tp = tile + (key >> 4) + ly * k3Pitch + 2 * (zb + ((q - zb) & 3));
#pragma unroll
                        for (int p = 0; p < 8; ++p) {
                            const float4 v = *reinterpret_cast<const float4*>(tp + p * k3Plane);
                            win[p][0] = make_float2(v.x, v.y);
                            win[p][1] = make_float2(v.z, v.w);
                        }
                    }
                    cur = key;
                }
                float2 t0 = __fmul2_rn(w3_dup(c.wa.x), win[0][0]), t1 = __fmul2_rn(w3_dup(c.wa.x), win[0][1]);
                t0 = __ffma2_rn(w3_dup(c.wa.y), win[1][0], t0); t1 = __ffma2_rn(w3_dup(c.wa.y), win[1][1], t1);
                t0 = __ffma2_rn(w3_dup(c.wa.z), win[2][0], t0); t1 = __ffma2_rn(w3_dup(c.wa.z), win[2][1], t1);
                t0 = __ffma2_rn(w3_dup(c.wa.w), win[3][0], t0); t1 = __ffma2_rn(w3_dup(c.wa.w), win[3][1], t1);
                t0 = __ffma2_rn(w3_dup(c.wb.x), win[4][0], t0); t1 = __ffma2_rn(w3_dup(c.wb.x), win[4][1], t1);
                t0 = __ffma2_rn(w3_dup(c.wb.y), win[5][0], t0); t1 = __ffma2_rn(w3_dup(c.wb.y), win[5][1], t1);
                t0 = __ffma2_rn(w3_dup(c.wb.z), win[6][0], t0); t1 = __ffma2_rn(w3_dup(c.wb.z), win[6][1], t1);
                t0 = __ffma2_rn(w3_dup(c.wb.w), win[7][0], t0); t1 = __ffma2_rn(w3_dup(c.wb.w), win[7][1], t1);
                part[j] = __ffma2_rn(w3_dup(c.w1 * c.w2.x), t0, __fmul2_rn(w3_dup(c.w1 * c.w2.y), t1));
            }
            // transposing reduction: after the five steps the four lanes 4 j .. 4 j + 3 hold the total of sample j
            {
                const bool up = lane & 16;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const float2 send = up ? part[j] : part[j + 4], keep = up ? part[j + 4] : part[j];
                    part[j] = make_float2(keep.x + __shfl_xor_sync(0xffffffffu, send.x, 16),
                                          keep.y + __shfl_xor_sync(0xffffffffu, send.y, 16));
                }
            }
            {
                const bool up = lane & 8;
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const float2 send = up ? part[j] : part[j + 2], keep = up ? part[j + 2] : part[j];
                    part[j] = make_float2(keep.x + __shfl_xor_sync(0xffffffffu, send.x, 8),
                                          keep.y + __shfl_xor_sync(0xffffffffu, send.y, 8));
                }
            }
            {
                const bool up = lane & 4;
                const float2 send = up ? part[0] : part[1], keep = up ? part[1] : part[0];
                part[0] = make_float2(keep.x + __shfl_xor_sync(0xffffffffu, send.x, 4),
                                      keep.y + __shfl_xor_sync(0xffffffffu, send.y, 4));
            }
            part[0].x += __shfl_xor_sync(0xffffffffu, part[0].x, 2);
            part[0].y += __shfl_xor_sync(0xffffffffu, part[0].y, 2);
            part[0].x += __shfl_xor_sync(0xffffffffu, part[0].x, 1);
            part[0].y += __shfl_xor_sync(0xffffffffu, part[0].y, 1);
            if (q == 0) {
                const int sj = s8 + ly;
                if (sj < cnt) {
                    const int m = __float_as_int(rec[sj * kW3Rec + 25]);
                    yb[m] = part[0];
                }
            }
        }
        __syncwarp();
    }
    if (!tile_ready) mbar_wait(bar, 0);     // a warp without samples still has to see the copies land before exit
}

// ------------------------------------------------------------------------------------------------------------
// V^H: G += w0 w1 w2 y, window accumulators in registers, flushed to the shared tile under a lock
// ------------------------------------------------------------------------------------------------------------
// Tile lock of a CTA with more than one warp.  Everything it orders is SHARED memory touched by warps of one SM: the
// shared-memory pipe executes a warp's LDS / STS / ATOMS in issue order, so the read-modify-writes of the critical section
// lie between the warp's own CAS and EXCH without a fence.  The asm clobbers stop the compiler from moving shared-memory
// accesses across the lock.  (Measured, config 4: 2 / 4 warps per CTA under this lock 0.363 / 0.481 ms against 0.315 ms for
// one warp per CTA and no lock -- with or without fences the shared tile does not pay; kW3GridWarps = 1 is the default.)
__device__ __forceinline__ void w3_lock(int* l, int lane) {
    if (lane == 0)
        while (atomicCAS(l, 0, 1) != 0) {}
    __syncwarp();
    asm volatile("" ::: "memory");
}
__device__ __forceinline__ void w3_unlock(int* l, int lane) {
    asm volatile("" ::: "memory");
    __syncwarp();
    if (lane == 0) atomicExch(l, 0);
}

template <int NW, bool TABLE>
__global__ void __launch_bounds__(NW * 32)
gridding_win_3d_kernel(SampleData s, GridGeom g, const WorkItem* __restrict__ items, const float2* __restrict__ y,
                       float2* __restrict__ grid, KernelPoly P, const __grid_constant__ CUtensorMap tmap, int use_tmap,
                       const float* __restrict__ w3rec) {
    constexpr int CH = TABLE ? 16 : 32;
    extern __shared__ __align__(1024) unsigned char w3smem[];
    float2* tile = reinterpret_cast<float2*>(w3smem);
    float* recs = reinterpret_cast<float*>(tile + k3Cells);
    int* lock = reinterpret_cast<int*>(recs + NW * 32 * kW3Rec);
    const WorkItem wi = items[blockIdx.x];
    const int b = blockIdx.y;
    int o[3];
    unpack_k0(wi.origin, o);
    const int K0 = g.K[0], K1 = g.K[1], K2 = g.K[2];
    for (int i = threadIdx.x; i < k3Cells / 2; i += blockDim.x)
        reinterpret_cast<float4*>(tile)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (threadIdx.x == 0) *lock = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ly = lane >> 2, q = lane & 3;
    float* rec = recs + warp * 32 * kW3Rec;
    const float2* __restrict__ yb = y + (int64_t)b * g.M;
    int wb, we;
    w3_share<NW>(wi, warp, wb, we);
    float2 acc[8][2];
#pragma unroll
    for (int p = 0; p < 8; ++p) { acc[p][0] = make_float2(0.f, 0.f); acc[p][1] = make_float2(0.f, 0.f); }
    int cur = -1;
    // flush the pairs that leave the window (all of them when `steps` is outside 1..3) and clear their accumulators
    auto retire = [&](int steps) {
        const int zc = cur & 15;
        const bool mine = (steps <= 0 || steps >= 4) || (((q - zc) & 3) < steps);
        if (NW > 1) w3_lock(lock, lane);
        if (mine) {
            float2* tp = tile + (cur >> 4) + ly * k3Pitch + 2 * (zc + ((q - zc) & 3));
#pragma unroll
            for (int p = 0; p < 8; ++p) {
                float4* cell = reinterpret_cast<float4*>(tp + p * k3Plane);
                float4 a = *cell;
                a.x += acc[p][0].x; a.y += acc[p][0].y; a.z += acc[p][1].x; a.w += acc[p][1].y;
                *cell = a;
                acc[p][0] = make_float2(0.f, 0.f);
                acc[p][1] = make_float2(0.f, 0.f);
            }
        }
        if (NW > 1) w3_unlock(lock, lane);
    };
    // two-deep prefetch: plan data of chunk c + 2 and the y values of chunk c + 1 are in flight while chunk c is applied
    W3Pre pre, nxt;
    uint64_t* wbar = reinterpret_cast<uint64_t*>(reinterpret_cast<unsigned char*>(lock) + 16) + 2 * warp;
    float* const rec0 = rec;
    // TABLE: only the caller's index and y are fetched through registers (two / one chunk ahead); the weights arrive by bulk copy
    auto fetch_m = [&](int si, bool valid, W3Pre& f) { f.m = valid ? __ldg(&s.perm[si]) : -1; f.yv = make_float2(0.f, 0.f); };
    if (TABLE) {
        if (lane == 0) {
            mbar_init(&wbar[0], 1);
            mbar_init(&wbar[1], 1);
            if (wb < we) {
                const int n0 = min(CH, we - wb);
                mbar_expect_tx(&wbar[0], (uint32_t)n0 * kW3Rec * 4);
                bulk_g2s(rec0, w3rec + (int64_t)wb * kW3Rec, (uint32_t)n0 * kW3Rec * 4, &wbar[0]);
            }
        }
        __syncwarp();
        fetch_m(wb + lane, lane < CH && wb + lane < we, pre);
        if (pre.m >= 0) pre.yv = __ldg(&yb[pre.m]);
        fetch_m(wb + CH + lane, lane < CH && wb + CH + lane < we, nxt);
    } else {
        w3_fetch(s, g, wb + lane, wb + lane < we, pre);
        if (pre.m >= 0) pre.yv = __ldg(&yb[pre.m]);
        w3_fetch(s, g, wb + 32 + lane, wb + 32 + lane < we, nxt);
    }
    int it = 0;
    for (int c0 = wb; c0 < we; c0 += CH, ++it) {
        const int cnt = min(CH, we - c0);
        if (TABLE) {
            rec = rec0 + (it & 1) * CH * kW3Rec;
            if (lane == 0 && c0 + CH < we) {
                const int n1 = min(CH, we - c0 - CH);
                fence_proxy_async_smem();         // this warp's y stores into that buffer precede the engine's writes
                mbar_expect_tx(&wbar[(it + 1) & 1], (uint32_t)n1 * kW3Rec * 4);
                bulk_g2s(rec0 + ((it + 1) & 1) * CH * kW3Rec, w3rec + (int64_t)(c0 + CH) * kW3Rec, (uint32_t)n1 * kW3Rec * 4,
                         &wbar[(it + 1) & 1]);
            }
            mbar_wait(&wbar[it & 1], (uint32_t)((it >> 1) & 1));
            if (lane < cnt) *reinterpret_cast<float2*>(rec + lane * kW3Rec + 26) = pre.yv;
            pre = nxt;
            if (pre.m >= 0) pre.yv = __ldg(&yb[pre.m]);
            fetch_m(c0 + 2 * CH + lane, lane < CH && c0 + 2 * CH + lane < we, nxt);
        } else {
            w3_stage(pre, g, P, o, rec + lane * kW3Rec);
            pre = nxt;
            if (pre.m >= 0) pre.yv = __ldg(&yb[pre.m]);
            w3_fetch(s, g, c0 + 64 + lane, c0 + 64 + lane < we, nxt);
        }
        __syncwarp();
        W3Rec nx = w3_load(rec, ly, q);
#pragma unroll 4
        for (int si = 0; si < cnt; ++si) {
            const W3Rec c = nx;
            nx = w3_load(rec + min(si + 1, CH - 1) * kW3Rec, ly, q);
            const int key = __float_as_int(c.kk.x);
            if (key != cur) {
                if (cur >= 0) retire(((key >> 4) == (cur >> 4)) ? (key & 15) - (cur & 15) : 4);
                cur = key;
            }
            const float l0 = c.w1 * c.w2.x, l1 = c.w1 * c.w2.y;
            const float2 v0 = make_float2(l0 * c.kk.z, l0 * c.kk.w), v1 = make_float2(l1 * c.kk.z, l1 * c.kk.w);
            acc[0][0] = __ffma2_rn(w3_dup(c.wa.x), v0, acc[0][0]); acc[0][1] = __ffma2_rn(w3_dup(c.wa.x), v1, acc[0][1]);
            acc[1][0] = __ffma2_rn(w3_dup(c.wa.y), v0, acc[1][0]); acc[1][1] = __ffma2_rn(w3_dup(c.wa.y), v1, acc[1][1]);
            acc[2][0] = __ffma2_rn(w3_dup(c.wa.z), v0, acc[2][0]); acc[2][1] = __ffma2_rn(w3_dup(c.wa.z), v1, acc[2][1]);
            acc[3][0] = __ffma2_rn(w3_dup(c.wa.w), v0, acc[3][0]); acc[3][1] = __ffma2_rn(w3_dup(c.wa.w), v1, acc[3][1]);
            acc[4][0] = __ffma2_rn(w3_dup(c.wb.x), v0, acc[4][0]); acc[4][1] = __ffma2_rn(w3_dup(c.wb.x), v1, acc[4][1]);
            acc[5][0] = __ffma2_rn(w3_dup(c.wb.y), v0, acc[5][0]); acc[5][1] = __ffma2_rn(w3_dup(c.wb.y), v1, acc[5][1]);
            acc[6][0] = __ffma2_rn(w3_dup(c.wb.z), v0, acc[6][0]); acc[6][1] = __ffma2_rn(w3_dup(c.wb.z), v1, acc[6][1]);
            acc[7][0] = __ffma2_rn(w3_dup(c.wb.w), v0, acc[7][0]); acc[7][1] = __ffma2_rn(w3_dup(c.wb.w), v1, acc[7][1]);
        }
        __syncwarp();
    }
    if (cur >= 0) retire(4);
    __syncthreads();
    // flush by the TMA engine: one bulk f32 reduce-add per padded row (rows wrap periodically; a row that crosses the
    // seam of the last axis is split); untouched cells are zeros and add nothing
    fence_proxy_async_smem();
    if (use_tmap && o[0] + k3P0 <= K0 && o[1] + k3P1 <= K1 && o[2] + k3Pitch <= K2) {
        __syncthreads();          // every thread's proxy fence precedes the one reduce
        if (threadIdx.x == 0) {
            tma_reduce_add_tile_4d(&tmap, 2 * o[2], o[1], o[0], b, tile);
            bulk_commit_and_wait_read();
        }
        return;
    }
    float2* __restrict__ Gb = grid + (int64_t)b * g.cells;
    for (int row = threadIdx.x; row < k3P0 * k3P1; row += blockDim.x) {
        const int lx = row / k3P1, lyy = row - lx * k3P1;
        const int gx = (o[0] + lx) & (K0 - 1), gy = (o[1] + lyy) & (K1 - 1), gz = o[2] & (K2 - 1);
        float2* dst = Gb + ((int64_t)gx * K1 + gy) * K2;
        const float2* src = tile + row * k3Pitch;
        const int first = min(k3Pitch, K2 - gz);
        bulk_s2g_add_f32(dst + gz, src, (uint32_t)first * 8);
        if (first < k3Pitch) bulk_s2g_add_f32(dst, src + first, (uint32_t)(k3Pitch - first) * 8);
    }
    bulk_commit_and_wait_read();
}

}  // namespace nufft
