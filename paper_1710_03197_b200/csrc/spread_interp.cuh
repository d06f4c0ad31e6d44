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
// J is a template parameter: widths other than kJ (SURVEY 8(f)-4 "other Jd") run on this kernel and on
// gridding_atomic_kernel below with a KernelPolyG.
// ------------------------------------------------------------------------------------------------------------
template <int D, int J = kJ, class Poly = KernelPoly>
__global__ void __launch_bounds__(128)
interp_direct_kernel(SampleData s, GridGeom g, const float2* __restrict__ grid, float2* __restrict__ y, Poly P) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.M) return;
    const int b = blockIdx.y;
    int k0[3];
    unpack_k0(__ldg(&s.kpack[i]), k0);
    float w[D][J];
#pragma unroll
    for (int a = 0; a < D; ++a) kb_weights_j<J>(P, a, __ldg(&s.delta[(int64_t)a * g.M + i]), w[a]);
    const float2* __restrict__ G = grid + (int64_t)b * g.cells;
    float2 acc = make_float2(0.f, 0.f);
    if (D == 1) {
        const int K0 = g.K[0];
#pragma unroll
        for (int j0 = 0; j0 < J; ++j0) {
            const float2 v = __ldg(&G[(k0[0] + j0) & (K0 - 1)]);
            acc.x = fmaf(w[0][j0], v.x, acc.x);
            acc.y = fmaf(w[0][j0], v.y, acc.y);
        }
    } else if (D == 2) {
        const int K0 = g.K[0], K1 = g.K[1];
#pragma unroll
        for (int j0 = 0; j0 < J; ++j0) {
            const float2* __restrict__ row = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1;
            float2 r = make_float2(0.f, 0.f);
#pragma unroll
            for (int j1 = 0; j1 < J; ++j1) {
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
        for (int j0 = 0; j0 < J; ++j0) {
            const float2* __restrict__ plane = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1 * K2;
            float2 rp = make_float2(0.f, 0.f);
#pragma unroll
            for (int j1 = 0; j1 < J; ++j1) {
                const float2* __restrict__ row = plane + (int64_t)((k0[1] + j1) & (K1 - 1)) * K2;
                float2 r = make_float2(0.f, 0.f);
#pragma unroll
                for (int j2 = 0; j2 < J; ++j2) {
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
template <int D, int J = kJ, class Poly = KernelPoly>
__global__ void __launch_bounds__(128)
gridding_atomic_kernel(SampleData s, GridGeom g, const float2* __restrict__ y, float2* __restrict__ grid, Poly P) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.M) return;
    const int b = blockIdx.y;
    int k0[3];
    unpack_k0(__ldg(&s.kpack[i]), k0);
    float w[D][J];
#pragma unroll
    for (int a = 0; a < D; ++a) kb_weights_j<J>(P, a, __ldg(&s.delta[(int64_t)a * g.M + i]), w[a]);
    const float2 yv = __ldg(&y[(int64_t)b * g.M + __ldg(&s.perm[i])]);
    float2* __restrict__ G = grid + (int64_t)b * g.cells;
    if (D == 1) {
        const int K0 = g.K[0];
#pragma unroll
        for (int j0 = 0; j0 < J; ++j0) atomicAdd(&G[(k0[0] + j0) & (K0 - 1)], cscale(yv, w[0][j0]));
    } else if (D == 2) {
        const int K0 = g.K[0], K1 = g.K[1];
#pragma unroll
        for (int j0 = 0; j0 < J; ++j0) {
            float2* __restrict__ row = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1;
            const float2 yr = cscale(yv, w[0][j0]);
#pragma unroll
            for (int j1 = 0; j1 < J; ++j1) atomicAdd(&row[(k0[1] + j1) & (K1 - 1)], cscale(yr, w[1][j1]));
        }
    } else {
        const int K0 = g.K[0], K1 = g.K[1], K2 = g.K[2];
#pragma unroll 1
        for (int j0 = 0; j0 < J; ++j0) {
            float2* __restrict__ plane = G + (int64_t)((k0[0] + j0) & (K0 - 1)) * K1 * K2;
            const float2 yp = cscale(yv, w[0][j0]);
#pragma unroll
            for (int j1 = 0; j1 < J; ++j1) {
                float2* __restrict__ row = plane + (int64_t)((k0[1] + j1) & (K1 - 1)) * K2;
                const float2 yr = cscale(yp, w[1][j1]);
#pragma unroll
                for (int j2 = 0; j2 < J; ++j2) atomicAdd(&row[(k0[2] + j2) & (K2 - 1)], cscale(yr, w[D - 1][j2]));
            }
        }
    }
}



// ============================================================================================================
// Tiled V^H (step a4): samples are sorted into grid tiles at plan time; a work item is (tile, sample range).  The
// padded tile (tile + J-1 halo cells per axis) is accumulated in shared memory WITHOUT atomics and flushed once.
//
// Shared-memory floating-point atomics are compare-and-swap loops on sm_100a (ATOMS.CAST.SPIN), so accumulation is
// organised so that no two warps ever touch the same cell:
//   2-D: every warp owns a private padded tile and walks its own work item sample by sample.  One sample is one
//        warp instruction group: lane (r, q), r = stencil row 0..5, q = 0..3, read-modify-writes the 16-byte pair of
//        cells q of row r of an 8-cell window aligned to an even column (24 active lanes, 3 + 3 wavefronts).
//   3-D: the six warps of a CTA share one padded tile; warp w handles, for every sample, the one stencil plane
//        whose tile-local index is = w (mod 6).  Planes of different warps are disjoint, so no synchronisation is
//        needed between samples.
// Weights are prepared 32 samples at a time, one sample per lane (kb_weights), and staged in shared memory as
//   rowrec[s][r] = (w_row * y.re, w_row * y.im, cell index of the window start of that row)      16 B
//   colrec[s][q] = the two column weights of cell pair q (0 outside the 6-cell support)          8 B
// so that the per-sample loop costs two small broadcast loads, one 16-byte RMW and four FMAs per lane.
// ============================================================================================================
struct WorkItem {
    uint32_t origin;     // tile origin per axis, packed like kpack
    int32_t s_begin;     // first sorted sample
    int32_t s_end;       // one past the last
    int32_t slab;        // deterministic mode: index of this item's private slab
};

struct TileGeom {
    int T[3];            // tile size per axis (cells)
    int P[3];            // padded extents: T + J - 1 (last axis rounded up to even = PITCH)
    int pitch;           // row pitch of the shared tile in cells (even)
    int plane;           // plane pitch in cells (3-D), P[1] * pitch
    int tile_cells;      // cells of one padded tile in shared memory
};

constexpr int kStageRow = 7;   // float4 slots per sample in rowrec (6 used; 7 keeps 8-lane phases conflict-free)
constexpr int kStageCol = 5;   // float2 slots per sample in colrec (4 used)
constexpr int kStageBytes = 32 * (kStageRow * 16 + kStageCol * 8);
// shared memory of one warp of gridding_tiled_2d_kernel: padded tile + staging, rounded up to 128 bytes
__host__ __device__ __forceinline__ int grid2d_warp_bytes(int tile_cells) { return ((tile_cells * 8 + kStageBytes + 127) / 128) * 128; }

// One lane prepares one sample of a 2-D work item.
__device__ __forceinline__ void stage_sample_2d(const KernelPoly& P, float4* rowrec, float2* colrec, int lane,
                                                int c0, int c1, float d0, float d1, float2 yv, int pitch, int base_off) {
    float w0[kJ], w1[kJ];
    kb_weights(P, 0, d0, w0);
    kb_weights(P, 1, d1, w1);
    const int par = c1 & 1, base = base_off + c0 * pitch + (c1 - par);
#pragma unroll
    for (int r = 0; r < kJ; ++r)
        rowrec[lane * kStageRow + r] = make_float4(w0[r] * yv.x, w0[r] * yv.y, __int_as_float(base + r * pitch), 0.f);
    colrec[lane * kStageCol + 0] = par ? make_float2(0.f, w1[0]) : make_float2(w1[0], w1[1]);
    colrec[lane * kStageCol + 1] = par ? make_float2(w1[1], w1[2]) : make_float2(w1[2], w1[3]);
    colrec[lane * kStageCol + 2] = par ? make_float2(w1[3], w1[4]) : make_float2(w1[4], w1[5]);
    colrec[lane * kStageCol + 3] = par ? make_float2(w1[5], 0.f) : make_float2(0.f, 0.f);
}

// Apply `cnt` staged samples to the shared tile: lane (r, q) handles cell pair q of stencil row r.
__device__ __forceinline__ void apply_staged(float2* tile, const float4* rowrec, const float2* colrec, int cnt, int lane) {
    if (lane >= 24) return;
    const int r = lane >> 2, q = lane & 3;
    for (int s = 0; s < cnt; ++s) {
        const float4 rr = rowrec[s * kStageRow + r];
        const float2 cc = colrec[s * kStageCol + q];
        float4* cell = reinterpret_cast<float4*>(tile + __float_as_int(rr.z) + 2 * q);
        float4 a = *cell;
        a.x = fmaf(rr.x, cc.x, a.x);
        a.y = fmaf(rr.y, cc.x, a.y);
        a.z = fmaf(rr.x, cc.y, a.z);
        a.w = fmaf(rr.y, cc.y, a.w);
        *cell = a;
    }
}

// Flush a padded tile: pair p of the shared tile goes to grid (atomic add) or to the item's private slab (store).
template <int D, bool DET>
__device__ __forceinline__ void flush_tile(const float2* tile, const TileGeom& tg, const GridGeom& g, uint32_t origin,
                                           float2* __restrict__ G, float2* __restrict__ slab, int tid, int nthreads) {
    int o[3];
    unpack_k0(origin, o);
    const int pairs_per_row = tg.pitch / 2;
    const int rows = (D == 2) ? tg.P[0] : tg.P[0] * tg.P[1];
    const int npairs = rows * pairs_per_row;
    for (int p = tid; p < npairs; p += nthreads) {
        const float4 v = reinterpret_cast<const float4*>(tile)[p];
        if (DET) {
            reinterpret_cast<float4*>(slab)[p] = v;
        } else {
            if (v.x == 0.f && v.y == 0.f && v.z == 0.f && v.w == 0.f) continue;
            const int row = p / pairs_per_row, cp = p - row * pairs_per_row;
            const int col = (o[D - 1] + 2 * cp) & (g.K[D - 1] - 1);
            int64_t gi;
            if (D == 2) {
                gi = (int64_t)((o[0] + row) & (g.K[0] - 1)) * g.K[1] + col;
            } else {
                const int lz = row / tg.P[1], ly = row - lz * tg.P[1];
                gi = ((int64_t)((o[0] + lz) & (g.K[0] - 1)) * g.K[1] + ((o[1] + ly) & (g.K[1] - 1))) * g.K[2] + col;
            }
            atomicAdd(reinterpret_cast<float4*>(G + gi), v);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Tiled V^H for any kernel width J in [kJmin, kJmax], 2-D (round 2; SURVEY 8(f)-4 "other Jd").  Same scheme as
// gridding_tiled_2d_kernel -- warp-private padded tile in shared memory, 32 samples staged at a time, one 16-byte
// read-modify-write per lane and sample, one TMA reduce-add flush per work item -- with the lane map derived from J:
// NP = (J + 2) / 2 cell pairs cover the (J + 1)-cell window aligned to an even column; a lane handles RPL stencil rows
// (J = 8: 5 pairs x 4 lane rows = 20 lanes, two rows each; J <= 7: one row per lane).  Replaces one global red.add per stencil point.
// ------------------------------------------------------------------------------------------------------------
template <int J> struct Tile2dJ {
    static constexpr int NP = (J + 2) / 2;
    static constexpr int RPL = (J + (32 / NP) - 1) / (32 / NP);      // stencil rows per lane (J = 8: 2, else 1)
    static constexpr int RL = (J + RPL - 1) / RPL;                  // lane rows: lane (rl, q) handles rows rl, rl + RL, ...
    static constexpr int ROWSLOTS = J | 1;            // float4 slots per sample (odd: 8-lane phases conflict-free)
    static constexpr int COLSLOTS = NP | 1;           // float2 slots per sample
    static constexpr int STAGE_BYTES = 32 * (ROWSLOTS * 16 + COLSLOTS * 8);
    __host__ __device__ static constexpr int warp_bytes(int tile_cells) { return ((tile_cells * 8 + STAGE_BYTES + 127) / 128) * 128; }
};

template <int J>
__global__ void __launch_bounds__(256)
gridding_tiled_2d_j_kernel(SampleData s, GridGeom g, TileGeom tg, const WorkItem* __restrict__ items, int n_items,
                           const float2* __restrict__ y, float2* __restrict__ grid, KernelPolyG P) {
    pdl_enter();
    using C = Tile2dJ<J>;
    extern __shared__ float4 smem4[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int item = blockIdx.x * nw + warp;
    if (item >= n_items) return;
    const int b = blockIdx.y;
    float2* tile = reinterpret_cast<float2*>(smem4 + (size_t)warp * (C::warp_bytes(tg.tile_cells) / 16));
    float4* rowrec = reinterpret_cast<float4*>(tile + tg.tile_cells);
    float2* colrec = reinterpret_cast<float2*>(rowrec + 32 * C::ROWSLOTS);
    const WorkItem wi = items[item];
    int o[3];
    unpack_k0(wi.origin, o);
    for (int i = lane; i < tg.tile_cells / 2; i += 32) reinterpret_cast<float4*>(tile)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncwarp();
    const float2* __restrict__ yb = y + (int64_t)b * g.M;
    for (int s0 = wi.s_begin; s0 < wi.s_end; s0 += 32) {
        const int si = s0 + lane;
        const int cnt = min(32, wi.s_end - s0);
        if (si < wi.s_end) {
            int k0[3];
            unpack_k0(__ldg(&s.kpack[si]), k0);
            float w0[J], w1[J];
            kb_weights_j<J>(P, 0, __ldg(&s.delta[si]), w0);
            kb_weights_j<J>(P, 1, __ldg(&s.delta[g.M + si]), w1);
            const float2 yv = __ldg(&yb[__ldg(&s.perm[si])]);
            const int c0 = (k0[0] - o[0]) & (g.K[0] - 1), c1 = (k0[1] - o[1]) & (g.K[1] - 1);
            const int par = c1 & 1, base = c0 * tg.pitch + (c1 - par);
#pragma unroll
            for (int r = 0; r < J; ++r)
                rowrec[lane * C::ROWSLOTS + r] = make_float4(w0[r] * yv.x, w0[r] * yv.y, __int_as_float(base + r * tg.pitch), 0.f);
#pragma unroll
            for (int q = 0; q < C::NP; ++q) {       // pair q = columns 2 q, 2 q + 1 of the aligned window = weights 2 q - par, + 1
                const int ja = 2 * q - par, jb = ja + 1;
                float wa = 0.f, wb = 0.f;
#pragma unroll
                for (int j = 0; j < J; ++j) { wa = (j == ja) ? w1[j] : wa; wb = (j == jb) ? w1[j] : wb; }
                colrec[lane * C::COLSLOTS + q] = make_float2(wa, wb);
            }
        }
        __syncwarp();
        {
            const int rl = lane / C::NP, q = lane % C::NP;
            if (lane < C::RL * C::NP) {
                for (int t = 0; t < cnt; ++t) {
                    const float2 cc = colrec[t * C::COLSLOTS + q];
#pragma unroll
                    for (int i = 0; i < C::RPL; ++i) {
                        const int r = rl + i * C::RL;
                        if (r < J) {
                            const float4 rr = rowrec[t * C::ROWSLOTS + r];
                            float4* cell = reinterpret_cast<float4*>(tile + __float_as_int(rr.z) + 2 * q);
                            float4 a = *cell;
                            a.x = fmaf(rr.x, cc.x, a.x);
                            a.y = fmaf(rr.y, cc.x, a.y);
                            a.z = fmaf(rr.x, cc.y, a.z);
                            a.w = fmaf(rr.y, cc.y, a.w);
                            *cell = a;
                        }
                    }
                }
            }
            __syncwarp();
        }
    }
    // flush by the TMA engine: one bulk f32 reduce-add per padded row (split at the seam of axis 1)
    fence_proxy_async_smem();
    float2* __restrict__ Gb = grid + (int64_t)b * g.cells;
    for (int row = lane; row < tg.P[0]; row += 32) {
        const int gx = (o[0] + row) & (g.K[0] - 1), gz = o[1] & (g.K[1] - 1);
        float2* dst = Gb + (int64_t)gx * g.K[1];
        const float2* src = tile + row * tg.pitch;
        const int first = min(tg.pitch, g.K[1] - gz);
        bulk_s2g_add_f32(dst + gz, src, (uint32_t)first * 8);
        if (first < tg.pitch) bulk_s2g_add_f32(dst, src + first, (uint32_t)(tg.pitch - first) * 8);
    }
    bulk_commit_and_wait_read();
}

// grid = 0 as a kernel (not a memset node), so that it takes part in the programmatic-dependent-launch chain of a transform
__global__ void __launch_bounds__(256) grid_zero_kernel(float4* __restrict__ g4, int64_t n4) {
    pdl_enter();
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (int64_t)gridDim.x * blockDim.x)
        g4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// 2-D: NW independent warps per CTA, each with a private tile + staging area.
template <bool DET>
__global__ void __launch_bounds__(256)
gridding_tiled_2d_kernel(SampleData s, GridGeom g, TileGeom tg, const WorkItem* __restrict__ items, int n_items,
                         const float2* __restrict__ y, float2* __restrict__ grid, float2* __restrict__ slabs,
                         int64_t slab_batch_stride, KernelPoly P, const __grid_constant__ CUtensorMap tmap, int use_tmap) {
    pdl_enter();
    extern __shared__ float4 smem4[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int item = blockIdx.x * nw + warp;
    if (item >= n_items) return;
    const int b = blockIdx.y;
    const int per_warp4 = grid2d_warp_bytes(tg.tile_cells) / 16;          // 128-byte multiple: every warp's tile is TMA-aligned
    float2* tile = reinterpret_cast<float2*>(smem4 + (size_t)warp * per_warp4);
    float4* rowrec = reinterpret_cast<float4*>(tile + tg.tile_cells);
    float2* colrec = reinterpret_cast<float2*>(rowrec + 32 * kStageRow);
    const WorkItem wi = items[item];
    int o[3];
    unpack_k0(wi.origin, o);
    const float2* __restrict__ yb = y + (int64_t)b * g.M;
    // plan data of chunk c + 2 and y of chunk c + 1 travel through registers while chunk c is applied: a warp walks its item
    // alone, so an unhidden load is two DRAM round trips per 32 samples (the whole batch-1 adjoint was paced by them)
    struct Pre { uint32_t kp; float d0, d1; int m; float2 yv; };
    auto fetch = [&](int si, Pre& f) {
        f.m = -1; f.kp = 0; f.d0 = f.d1 = 0.f; f.yv = make_float2(0.f, 0.f);
        if (si < wi.s_end) {
            f.kp = __ldg(&s.kpack[si]); f.d0 = __ldg(&s.delta[si]); f.d1 = __ldg(&s.delta[g.M + si]); f.m = __ldg(&s.perm[si]);
        }
    };
    Pre cur, nxt;
    fetch(wi.s_begin + lane, cur);
    if (cur.m >= 0) cur.yv = __ldg(&yb[cur.m]);
    fetch(wi.s_begin + 32 + lane, nxt);
    for (int i = lane; i < tg.tile_cells / 2; i += 32) reinterpret_cast<float4*>(tile)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncwarp();
    for (int s0 = wi.s_begin; s0 < wi.s_end; s0 += 32) {
        const int cnt = min(32, wi.s_end - s0);
        if (cur.m >= 0) {
            int k0[3];
            unpack_k0(cur.kp, k0);
            stage_sample_2d(P, rowrec, colrec, lane, (k0[0] - o[0]) & (g.K[0] - 1), (k0[1] - o[1]) & (g.K[1] - 1), cur.d0, cur.d1,
                            cur.yv, tg.pitch, 0);
        }
        cur = nxt;
        if (cur.m >= 0) cur.yv = __ldg(&yb[cur.m]);
        fetch(s0 + 64 + lane, nxt);
        __syncwarp();
        apply_staged(tile, rowrec, colrec, cnt, lane);
        __syncwarp();
    }
    if (!DET) {       // flush by the TMA engine: one bulk f32 reduce-add per padded row (split at the seam of axis 1)
        fence_proxy_async_smem();
        if (use_tmap && o[0] + tg.P[0] <= g.K[0] && o[1] + tg.pitch <= g.K[1]) {      // one tensor-map reduce-add per item
            __syncwarp();
            if (lane == 0) {
                tma_reduce_add_tile_3d(&tmap, 2 * o[1], o[0], b, tile);
                bulk_commit_and_wait_read();
            }
            return;
        }
        float2* __restrict__ Gb = grid + (int64_t)b * g.cells;
        for (int row = lane; row < tg.P[0]; row += 32) {
            const int gx = (o[0] + row) & (g.K[0] - 1), gz = o[1] & (g.K[1] - 1);
            float2* dst = Gb + (int64_t)gx * g.K[1];
            const float2* src = tile + row * tg.pitch;
            const int first = min(tg.pitch, g.K[1] - gz);
            bulk_s2g_add_f32(dst + gz, src, (uint32_t)first * 8);
            if (first < tg.pitch) bulk_s2g_add_f32(dst, src + first, (uint32_t)(tg.pitch - first) * 8);
        }
        bulk_commit_and_wait_read();
        return;
    }
    flush_tile<2, DET>(tile, tg, g, wi.origin, grid + (int64_t)b * g.cells,
                       DET ? slabs + (int64_t)b * slab_batch_stride + (int64_t)wi.slab * tg.tile_cells : nullptr, lane, 32);
}

// 3-D: one work item per CTA of 6 warps; warp w owns the tile-local planes = w (mod 6).
// Staging is CTA-wide, 32 samples per round: warp 0 writes the part every warp needs (per stencil row r: the row weight
// and the cell offset of the row's 8-cell window; per cell pair q: the two column weights), every warp writes its own
// 16 bytes per sample (y times the plane weight of ITS plane of that sample, and the plane offset).  Per sample and
// warp the apply loop then costs three small loads, one 16-byte read-modify-write and six FMAs per lane.
constexpr int k3CommonF2 = 10;                                             // float2 slots per sample: 6 rows + 4 pairs
constexpr int kStage3dBytes = 32 * k3CommonF2 * 8 + 6 * 32 * 16;           // 2560 + 3072

template <bool DET>
__global__ void __launch_bounds__(192)
gridding_tiled_3d_kernel(SampleData s, GridGeom g, TileGeom tg, const WorkItem* __restrict__ items, int n_items,
                         const float2* __restrict__ y, float2* __restrict__ grid, float2* __restrict__ slabs,
                         int64_t slab_batch_stride, KernelPoly P) {
    extern __shared__ float4 smem4[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y;
    float2* tile = reinterpret_cast<float2*>(smem4);
    float2* common = tile + tg.tile_cells;                                  // [32][k3CommonF2]
    float4* perwarp = reinterpret_cast<float4*>(common + 32 * k3CommonF2);  // [6][32]
    const WorkItem wi = items[blockIdx.x];
    int o[3];
    unpack_k0(wi.origin, o);
    for (int i = threadIdx.x; i < tg.tile_cells / 2; i += blockDim.x)
        reinterpret_cast<float4*>(tile)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    const float2* __restrict__ yb = y + (int64_t)b * g.M;
    const int r = lane >> 2, q = lane & 3;
    for (int s0 = wi.s_begin; s0 < wi.s_end; s0 += 32) {
        const int si = s0 + lane;
        const int cnt = min(32, wi.s_end - s0);
        __syncthreads();              // tile zeroed (first round) / previous round's records consumed
        if (si < wi.s_end) {
            int k0[3];
            unpack_k0(__ldg(&s.kpack[si]), k0);
            const float2 yv = __ldg(&yb[__ldg(&s.perm[si])]);
            const int c0 = (k0[0] - o[0]) & (g.K[0] - 1);
            // this warp's plane of the sample: tile-local plane c0 + j0 = warp (mod 6)
            const int j0 = (warp - c0 % 6 + 6) % 6;
            float wz[kJ];
            kb_weights(P, 0, __ldg(&s.delta[si]), wz);
            float wsel = wz[0];
#pragma unroll
            for (int j = 1; j < kJ; ++j) wsel = (j0 == j) ? wz[j] : wsel;
            perwarp[warp * 32 + lane] = make_float4(yv.x * wsel, yv.y * wsel, __int_as_float((c0 + j0) * tg.plane), 0.f);
            if (warp == 0) {
                const int c1 = (k0[1] - o[1]) & (g.K[1] - 1), c2 = (k0[2] - o[2]) & (g.K[2] - 1);
                float w1[kJ], w2[kJ];
                kb_weights(P, 1, __ldg(&s.delta[g.M + si]), w1);
                kb_weights(P, 2, __ldg(&s.delta[2 * g.M + si]), w2);
                const int par = c2 & 1, base = c1 * tg.pitch + (c2 - par);
                float2* rec = common + lane * k3CommonF2;
#pragma unroll
                for (int rr = 0; rr < kJ; ++rr) rec[rr] = make_float2(w1[rr], __int_as_float(base + rr * tg.pitch));
                rec[6] = par ? make_float2(0.f, w2[0]) : make_float2(w2[0], w2[1]);
                rec[7] = par ? make_float2(w2[1], w2[2]) : make_float2(w2[2], w2[3]);
                rec[8] = par ? make_float2(w2[3], w2[4]) : make_float2(w2[4], w2[5]);
                rec[9] = par ? make_float2(w2[5], 0.f) : make_float2(0.f, 0.f);
            }
        }
        __syncthreads();
        if (lane < 24) {
            // Run-length merge: consecutive samples of the sorted order that share all three stencil base indices (a
            // radial readout oversampled 2x advances half a cell per sample) hit the same cells; their contributions
            // are summed in registers and written with ONE read-modify-write.  The test is warp-uniform.
            const float4* pw = perwarp + warp * 32;
            int prevkey = -1;
            float4 pend = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int sidx = 0; sidx < cnt; ++sidx) {
                const float4 ps = pw[sidx];
                const float2 wr = common[sidx * k3CommonF2 + r];
                const float2 cc = common[sidx * k3CommonF2 + 6 + q];
                const float rx = ps.x * wr.x, ry = ps.y * wr.x;
                const int key = __float_as_int(ps.z) + __float_as_int(wr.y);
                if (key != prevkey) {
                    if (prevkey >= 0) {
                        float4* cell = reinterpret_cast<float4*>(tile + prevkey + 2 * q);
                        float4 a = *cell;
                        a.x += pend.x; a.y += pend.y; a.z += pend.z; a.w += pend.w;
                        *cell = a;
                    }
                    pend = make_float4(0.f, 0.f, 0.f, 0.f);
                    prevkey = key;
                }
                pend.x = fmaf(rx, cc.x, pend.x);
                pend.y = fmaf(ry, cc.x, pend.y);
                pend.z = fmaf(rx, cc.y, pend.z);
                pend.w = fmaf(ry, cc.y, pend.w);
            }
            if (prevkey >= 0) {
                float4* cell = reinterpret_cast<float4*>(tile + prevkey + 2 * q);
                float4 a = *cell;
                a.x += pend.x; a.y += pend.y; a.z += pend.z; a.w += pend.w;
                *cell = a;
            }
        }
    }
    __syncthreads();
    if (!DET && tg.pitch * 8 % 16 == 0) {
        // flush by the TMA engine: one bulk f32 reduce-add per padded row (rows wrap periodically; a row that crosses the
        // seam of the last axis is split); the tile's untouched cells are zeros and add nothing
        fence_proxy_async_smem();
        float2* __restrict__ Gb = grid + (int64_t)b * g.cells;
        const int rows = tg.P[0] * tg.P[1];
        for (int row = threadIdx.x; row < rows; row += blockDim.x) {
            const int lx = row / tg.P[1], ly = row - lx * tg.P[1];
            const int gx = (o[0] + lx) & (g.K[0] - 1), gy = (o[1] + ly) & (g.K[1] - 1), gz = o[2] & (g.K[2] - 1);
            float2* dst = Gb + ((int64_t)gx * g.K[1] + gy) * g.K[2];
            const float2* src = tile + row * tg.pitch;
            const int first = min(tg.pitch, g.K[2] - gz);
            bulk_s2g_add_f32(dst + gz, src, (uint32_t)first * 8);
            if (first < tg.pitch) bulk_s2g_add_f32(dst, src + first, (uint32_t)(tg.pitch - first) * 8);
        }
        bulk_commit_and_wait_read();      // shared memory must stay valid until the engine has read it
        return;
    }
    flush_tile<3, DET>(tile, tg, g, wi.origin, grid + (int64_t)b * g.cells,
                       DET ? slabs + (int64_t)b * slab_batch_stride + (int64_t)wi.slab * tg.tile_cells : nullptr,
                       threadIdx.x, blockDim.x);
}

// Deterministic merge: every grid cell sums, in fixed order, the slabs of the work items whose padded tile covers it.
// tile_item_start[t] .. tile_item_start[t+1] are the slabs of tile t (work items of one tile are contiguous).
template <int D>
__global__ void __launch_bounds__(256)
gridding_merge_kernel(GridGeom g, TileGeom tg, int nt0, int nt1, int nt2, const int32_t* __restrict__ tile_item_start,
                      const float2* __restrict__ slabs, int64_t slab_batch_stride, float2* __restrict__ grid) {
    const int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= g.cells) return;
    const int b = blockIdx.y;
    int c[3];
    if (D == 2) { c[0] = (int)(cell / g.K[1]); c[1] = (int)(cell % g.K[1]); c[2] = 0; }
    else { c[2] = (int)(cell % g.K[2]); const int64_t q = cell / g.K[2]; c[1] = (int)(q % g.K[1]); c[0] = (int)(q / g.K[1]); }
    const int nt[3] = {nt0, nt1, nt2};
    // per axis: the tile containing the cell, and (if the cell lies in the first J-1 cells of it) the previous tile
    int t[3][2], l[3][2], n[3];
#pragma unroll
    for (int a = 0; a < D; ++a) {
        const int ti = c[a] / tg.T[a], li = c[a] - ti * tg.T[a];
        // previous tile first (fixed order): its local index is li + T
        n[a] = 0;
        if (li < kJ - 1) {
            t[a][n[a]] = (ti + nt[a] - 1) % nt[a]; l[a][n[a]] = li + tg.T[a]; n[a]++;
        }
        t[a][n[a]] = ti; l[a][n[a]] = li; n[a]++;
    }
    const float2* __restrict__ S = slabs + (int64_t)b * slab_batch_stride;
    float2 acc = make_float2(0.f, 0.f);
    for (int i0 = 0; i0 < n[0]; ++i0)
        for (int i1 = 0; i1 < n[1]; ++i1)
            for (int i2 = 0; i2 < (D == 3 ? n[2] : 1); ++i2) {
                int tid_, off;
                if (D == 2) { tid_ = t[0][i0] * nt1 + t[1][i1]; off = l[0][i0] * tg.pitch + l[1][i1]; }
                else { tid_ = (t[0][i0] * nt1 + t[1][i1]) * nt2 + t[2][i2]; off = l[0][i0] * tg.plane + l[1][i1] * tg.pitch + l[2][i2]; }
                for (int w = tile_item_start[tid_]; w < tile_item_start[tid_ + 1]; ++w)
                    acc = cadd(acc, S[(int64_t)w * tg.tile_cells + off]);
            }
    grid[(int64_t)b * g.cells + cell] = acc;
}
// ------------------------------------------------------------------------------------------------------------
// V, 2-D planar, tile-staged (round 2; small batches): one CTA per work item (tile, sample range), one thread per sample.
// profiles/r01b: with the direct form every warp load touches ~16 sectors and the L1 data pipe saturates; here the padded
// tile of the item (default 21 x 40 cells = 6.7 KB) is staged in shared memory with one bulk copy per row and the 36
// stencil values of a sample are 36 shared-memory loads.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
interp_tiled_2d_kernel(SampleData s, GridGeom g, TileGeom tg, const WorkItem* __restrict__ items,
                       const float2* __restrict__ grid, float2* __restrict__ y, KernelPoly P,
                       const __grid_constant__ CUtensorMap tmap, int use_tmap) {
    pdl_enter();
    extern __shared__ float4 smem4[];
    float2* tile = reinterpret_cast<float2*>(smem4);
    uint64_t* bar = reinterpret_cast<uint64_t*>(tile + tg.tile_cells);
    const WorkItem wi = items[blockIdx.x];
    const int b = blockIdx.y;
    int o[3];
    unpack_k0(wi.origin, o);
    const int K0 = g.K[0], K1 = g.K[1];
    const float2* __restrict__ G = grid + (int64_t)b * g.cells;
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_expect_tx(bar, (uint32_t)(tg.P[0] * tg.pitch * 8));
    }
    __syncthreads();
    if (use_tmap && o[0] + tg.P[0] <= K0 && o[1] + tg.pitch <= K1) {      // one tensor-map copy for the whole padded tile
        if (threadIdx.x == 0) tma_load_tile_3d(tile, &tmap, 2 * o[1], o[0], b, bar);
    } else {                                                              // seam tiles: one bulk copy per row, split at the seam
        for (int row = threadIdx.x; row < tg.P[0]; row += blockDim.x) {
            const int gx = (o[0] + row) & (K0 - 1), gz = o[1] & (K1 - 1);
            const float2* src = G + (int64_t)gx * K1;
            float2* dst = tile + row * tg.pitch;
            const int first = min(tg.pitch, K1 - gz);
            bulk_g2s(dst, src + gz, (uint32_t)first * 8, bar);
            if (first < tg.pitch) bulk_g2s(dst + first, src, (uint32_t)(tg.pitch - first) * 8, bar);
        }
    }
    // the sample's plan data and weights are fetched / evaluated while the copies are in flight
    float2* __restrict__ yb = y + (int64_t)b * g.M;
    for (int base = wi.s_begin; base < wi.s_end; base += blockDim.x) {
        const int si = base + threadIdx.x;
        const bool valid = si < wi.s_end;
        int k0[3] = {0, 0, 0};
        float w0[kJ], w1[kJ];
        int m = 0;
        if (valid) {
            unpack_k0(__ldg(&s.kpack[si]), k0);
            kb_weights(P, 0, __ldg(&s.delta[si]), w0);
            kb_weights(P, 1, __ldg(&s.delta[g.M + si]), w1);
            m = __ldg(&s.perm[si]);
        }
        if (base == wi.s_begin) mbar_wait(bar, 0);
        if (!valid) continue;
        const float2* __restrict__ tp = tile + ((k0[0] - o[0]) & (K0 - 1)) * tg.pitch + ((k0[1] - o[1]) & (K1 - 1));
        float2 acc = make_float2(0.f, 0.f);
#pragma unroll
        for (int j0 = 0; j0 < kJ; ++j0) {
            float2 r = make_float2(0.f, 0.f);
#pragma unroll
            for (int j1 = 0; j1 < kJ; ++j1) {
                const float2 v = tp[j0 * tg.pitch + j1];
                r.x = fmaf(w1[j1], v.x, r.x);
                r.y = fmaf(w1[j1], v.y, r.y);
            }
            acc.x = fmaf(w0[j0], r.x, acc.x);
            acc.y = fmaf(w0[j0], r.y, acc.y);
        }
        yb[m] = acc;
    }
}

}  // namespace nufft

namespace nufft {
// ============================================================================================================
// Tiled V, 3-D (step a3), batch 1.  profiles/r01b + the 3-D capture: with one thread per sample every load
// instruction of a warp touches ~16 sectors in as many lines and the L1 data pipe saturates (l1tex 98 %).  Here a CTA
// owns one work item (tile 8 x 8 x 16 cells + halo, sample range): it stages the padded tile (13 x 13 x 24 cells,
// 32 KB) in shared memory with coalesced 16-byte loads and then every HALF-WARP interpolates one sample: lane
// (rr, cc) reads cell (row 2g + rr, column cc) of an 8-cell window of stencil plane p -- two 64-byte row segments per
// half-warp load, bank-conflict free because the row pitch is 8 (mod 16) cells -- 18 loads per sample pair instead
// of 216 per sample, then a 4-step shuffle reduction.  Weights: one thread per sample evaluates kb_weights and parks
// w0[6], w1[6], w2[6] (zero-padded to 8) in shared memory.
// ============================================================================================================
constexpr int k3T0 = 8, k3T1 = 8, k3T2 = 16;
constexpr int k3P0 = k3T0 + kJ - 1, k3P1 = k3T1 + kJ - 1;      // 13 x 13 padded rows
constexpr int k3Pitch = 24;                                    // cells per padded row (8 mod 16), >= 16 + 5 + 2
constexpr int k3Plane = k3P1 * k3Pitch;
constexpr int k3Cells = k3P0 * k3Plane;                        // 4056 cells = 32448 B
constexpr int k3Chunk = 128;                                   // samples whose weights are staged at a time
constexpr int k3RecW = 28;                                     // floats per staged sample record
constexpr int kInterp3dSmem = k3Cells * 8 + k3Chunk * k3RecW * 4 + 16;

__global__ void __launch_bounds__(256)
interp_tiled_3d_kernel(SampleData s, GridGeom g, const WorkItem* __restrict__ items, const float2* __restrict__ grid,
                       float2* __restrict__ y, KernelPoly P) {
    extern __shared__ float4 smem4[];
    float2* tile = reinterpret_cast<float2*>(smem4);
    float* recs = reinterpret_cast<float*>(tile + k3Cells);
    const WorkItem wi = items[blockIdx.x];
    const int b = blockIdx.y;
    int o[3];
    unpack_k0(wi.origin, o);
    const int K0 = g.K[0], K1 = g.K[1], K2 = g.K[2];
    const float2* __restrict__ G = grid + (int64_t)b * g.cells;
    // stage the padded tile with bulk copies (cp.async.bulk + mbarrier, SASS UBLKCP): one 192-byte row (24 cells) per
    // thread, rows wrap periodically, a row that crosses the seam of the last axis is split in two copies
    uint64_t* bar = reinterpret_cast<uint64_t*>(recs + k3Chunk * k3RecW);
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        mbar_expect_tx(bar, (uint32_t)(k3P0 * k3P1 * k3Pitch * 8));
    }
    __syncthreads();
    for (int row = threadIdx.x; row < k3P0 * k3P1; row += blockDim.x) {
        const int lx = row / k3P1, ly = row - lx * k3P1;
        const int gx = (o[0] + lx) & (K0 - 1), gy = (o[1] + ly) & (K1 - 1), gz = o[2] & (K2 - 1);
        const float2* src = G + ((int64_t)gx * K1 + gy) * K2;
        float2* dst = tile + row * k3Pitch;
        const int first = min(k3Pitch, K2 - gz);
        bulk_g2s(dst, src + gz, (uint32_t)first * 8, bar);
        if (first < k3Pitch) bulk_g2s(dst + first, src, (uint32_t)(k3Pitch - first) * 8, bar);
    }
    mbar_wait(bar, 0);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int half = lane >> 4, rr = (lane >> 3) & 1, cc = lane & 7;
    const int lane_off = rr * k3Pitch + cc;
    float2* __restrict__ yb = y + (int64_t)b * g.M;
    for (int c0 = wi.s_begin; c0 < wi.s_end; c0 += k3Chunk) {
        const int cnt = min(k3Chunk, wi.s_end - c0);
        __syncthreads();          // tile staged (first pass) / previous chunk's records consumed
        for (int t = threadIdx.x; t < cnt; t += blockDim.x) {
            const int si = c0 + t;
            int k0[3];
            unpack_k0(__ldg(&s.kpack[si]), k0);
            float w0[kJ], w1[kJ], w2[kJ];
            kb_weights(P, 0, __ldg(&s.delta[si]), w0);
            kb_weights(P, 1, __ldg(&s.delta[g.M + si]), w1);
            kb_weights(P, 2, __ldg(&s.delta[2 * g.M + si]), w2);
            float4* r = reinterpret_cast<float4*>(recs + t * k3RecW);
            r[0] = make_float4(w0[0], w0[1], w0[2], w0[3]);
            r[1] = make_float4(w0[4], w0[5], 0.f, 0.f);
            r[2] = make_float4(w1[0], w1[1], w1[2], w1[3]);
            r[3] = make_float4(w1[4], w1[5], 0.f, 0.f);
            r[4] = make_float4(w2[0], w2[1], w2[2], w2[3]);
            r[5] = make_float4(w2[4], w2[5], 0.f, 0.f);
            const int l0 = (k0[0] - o[0]) & (K0 - 1), l1 = (k0[1] - o[1]) & (K1 - 1), l2 = (k0[2] - o[2]) & (K2 - 1);
            r[6] = make_float4(__int_as_float(l0 * k3Plane + l1 * k3Pitch + l2), __int_as_float(__ldg(&s.perm[si])), 0.f, 0.f);
        }
        __syncthreads();
        // half-warp per sample; a warp handles sample pairs warp*2 + half, + 16, ...
        for (int t0 = warp * 2; t0 < cnt; t0 += 16) {
            const int t = t0 + half;
            const bool valid = t < cnt;
            const float* rec = recs + (valid ? t : t0) * k3RecW;
            const float4 wa = *reinterpret_cast<const float4*>(rec), wb = *reinterpret_cast<const float4*>(rec + 4);
            const float w0[kJ] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y};
            const float wc = rec[16 + cc];
            // packed two-wide FP32 FMA (fma.rn.f32x2 / FFMA2): (re, im) of a cell travel as one register pair
            const float wa0 = rec[8 + rr] * wc, wa1 = rec[10 + rr] * wc, wa2 = rec[12 + rr] * wc;
            const float2 w12[3] = {make_float2(wa0, wa0), make_float2(wa1, wa1), make_float2(wa2, wa2)};
            const float2* __restrict__ tp = tile + __float_as_int(rec[24]) + lane_off;
            float2 acc = make_float2(0.f, 0.f);
#pragma unroll
            for (int p = 0; p < kJ; ++p) {
                float2 tsum = __fmul2_rn(w12[0], tp[p * k3Plane]);
                tsum = __ffma2_rn(w12[1], tp[p * k3Plane + 2 * k3Pitch], tsum);
                tsum = __ffma2_rn(w12[2], tp[p * k3Plane + 4 * k3Pitch], tsum);
                acc = __ffma2_rn(make_float2(w0[p], w0[p]), tsum, acc);
            }
#pragma unroll
            for (int off = 8; off > 0; off >>= 1) {
                acc.x += __shfl_xor_sync(0xffffffffu, acc.x, off);
                acc.y += __shfl_xor_sync(0xffffffffu, acc.y, off);
            }
            if (valid && (lane & 15) == 0) yb[__float_as_int(rec[25])] = acc;
        }
    }
}
}  // namespace nufft
