// batch_il.cuh -- the batch-interleaved 2-D path (steps a1..a6 and a8 of SURVEY.md 8(a) for batches >= 12 images that
// share one trajectory: the paper's batch mode PAPER.md:52 and the multi-coil operator PAPER.md:251-258).
//
// Why a second layout.  At J = 6 every sample touches 36 complex64 grid cells; with a planar grid and one thread per
// sample that is 36 loads of ~21 sectors per warp and the L1 data pipe saturates (profiles/r01b: l1tex 96 %).  Here
// the workspace grid is stored as  grid_il[group][K0][K1][32]  (32 images of a group side by side, 256 contiguous
// bytes per grid cell) and LANES ARE IMAGES: one warp load fetches one stencil point of 32 images as two full 128-B
// lines, interpolation weights are warp-uniform, and nothing is gathered per lane.
//
//   F   rows: fft_il_rows_{fwd,adj}_kernel  planar image <-> interleaved grid (S, zero-pad / crop, coil multiply fused)
//       cols: the generic strided pass fft_cols_kernel over [K0][K1*32]
//   V   interp_il_kernel     one warp = 32 consecutive cell-sorted samples x 32 images
//   V^H gridding_il_kernel   GATHER form, accumulation in REGISTERS: warp = one grid row x 8 columns x 32 images;
//                            it walks the samples whose stencil covers that row (contiguous ranges of the
//                            cell-sorted order, found through rowptr) and adds w0 * w1 * y.  No atomics, no
//                            shared-memory read-modify-write, no zero-fill; every grid cell is written exactly once,
//                            in a fixed summation order (bit-reproducible).  The contiguous table / sample ranges
//                            of a CTA are staged in shared memory by bulk copies (cp.async.bulk + mbarrier).
#pragma once
#include "common.cuh"
#include "fft.cuh"
#include "spread_interp.cuh"

namespace nufft {

constexpr int kIL = 32;      // images per interleaved group (= lanes per warp)
constexpr int kBandW = 8;    // grid columns per V^H band (accumulators per lane: kBandW complex)
constexpr int kTabW = 24;    // floats per sample in the V^H weight table: w0 rotated [8], w1 band-aligned A[8], B[8]

// ------------------------------------------------------------------------------------------------------------
// FFT row passes between the caller's planar images and the interleaved grid
// ------------------------------------------------------------------------------------------------------------
struct IlRowParams {
    const float2* img_in;     // forward: x [batch][N0][N1]
    float2* img_out;          // adjoint: x [batch][N0][N1]
    float2* grid;             // grid_il [groups][K0][K1][32]
    const float2* coil;       // optional [batch][N0][N1]
    const float* s_outer;     // scaling vector of axis 0 (length N0)
    const float* s_line;      // scaling vector of axis 1 (length N1)
    const float2* tw;         // twiddles of length K1
    int n_outer, k_outer;     // N0, K0
    int batch;                // images present (lanes >= batch of the last group are idle)
    int same_image;           // forward: every batch item reads image 0 (multi-coil forward)
};

// a1 + first pass of a2: x (scaled, circularly zero-padded) -> FFT along axis 1 -> grid_il rows
// CTA = T images of one image row; thread (t, q0) works on image t.
template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::TS, (K == 512) ? 4 : 1)
fft_il_rows_fwd_kernel(IlRowParams p) {
    pdl_enter();
    constexpr int N = K / 2, T = Rad<K>::TS;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, q0 = threadIdx.x / T;
    const int n0 = blockIdx.x % p.n_outer;
    const int b = (blockIdx.x / p.n_outer) * T + t;
    const bool active = b < p.batch;
    const int bb = active ? b : 0;
    const int g0 = (n0 - p.n_outer / 2) & (p.k_outer - 1);
    const float2* __restrict__ src = p.img_in + ((int64_t)(p.same_image ? 0 : bb) * p.n_outer + n0) * N;
    const float2* __restrict__ csrc = p.coil ? p.coil + ((int64_t)bb * p.n_outer + n0) * N : nullptr;
    float2* __restrict__ dst = p.grid + (((int64_t)(b / kIL) * p.k_outer + g0) * K) * kIL + (b % kIL);
    const float so = __ldg(&p.s_outer[n0]);
    const float* __restrict__ sl = p.s_line;
    LayStrided<K, T> lay{smem + t};
    auto ld = [&](int i) -> float2 {
        const int n = (i + N / 2) & (K - 1);
        float2 xv = __ldg(&src[n]);
        if (csrc) xv = cmul(xv, __ldg(&csrc[n]));
        return cscale(xv, so * __ldg(&sl[n]));
    };
    auto st = [&](int i, float2 v) { dst[(int64_t)i * kIL] = v; };
    fft_line<K, true, false>(q0, active, lay, p.tw, ld, st);
}

// last pass of a5 + a6: grid_il rows -> inverse FFT along axis 1 -> crop -> S^H (-> conj(coil)) -> planar images
template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::TS)
fft_il_rows_adj_kernel(IlRowParams p) {
    pdl_enter();
    constexpr int N = K / 2, T = Rad<K>::TS;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, q0 = threadIdx.x / T;
    const int n0 = blockIdx.x % p.n_outer;
    const int b = (blockIdx.x / p.n_outer) * T + t;
    const bool active = b < p.batch;
    const int bb = active ? b : 0;
    const int g0 = (n0 - p.n_outer / 2) & (p.k_outer - 1);
    const float2* __restrict__ src = p.grid + (((int64_t)(b / kIL) * p.k_outer + g0) * K) * kIL + (b % kIL);
    float2* __restrict__ dst = p.img_out + ((int64_t)bb * p.n_outer + n0) * N;
    const float2* __restrict__ csrc = p.coil ? p.coil + ((int64_t)bb * p.n_outer + n0) * N : nullptr;
    const float so = __ldg(&p.s_outer[n0]);
    const float* __restrict__ sl = p.s_line;
    LayStrided<K, T> lay{smem + t};
    auto ld = [&](int i) -> float2 { return cconj(src[(int64_t)i * kIL]); };
    auto st = [&](int i, float2 v) {
        const int n = (i + N / 2) & (K - 1);
        float2 r = cscale(cconj(v), so * __ldg(&sl[n]));
        if (csrc) r = cmul(r, cconj(__ldg(&csrc[n])));
        dst[n] = r;
    };
    fft_line<K, false, true>(q0, active, lay, p.tw, ld, st);
}

// Multi-coil variant of the pass above with the coil sum of eq. (35) fused: x[n] = sum_i conj(c_i[n]) (S^H F^H grid_i)[n].
// CTA = one image row; it walks the coils T at a time (thread (t, q0) works on coil o T + t), multiplies by conj(c_i),
// sums the T coils of an octet with lane shuffles (the T lanes of a q0 are adjacent) and keeps the running sum over the
// octets in registers: the per-coil images are never written, coil_sum_kernel is not needed, the order is fixed.
template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::TS)
fft_il_rows_adj_coilsum_kernel(IlRowParams p) {
    pdl_enter();
    constexpr int N = K / 2, T = Rad<K>::TS, E = Rad<K>::E;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, q0 = threadIdx.x / T;
    const int n0 = blockIdx.x;
    const int g0 = (n0 - p.n_outer / 2) & (p.k_outer - 1);
    const float so = __ldg(&p.s_outer[n0]);
    const float* __restrict__ sl = p.s_line;
    LayStrided<K, T> lay{smem + t};
    float2 acc[E];
    int nidx[E];
#pragma unroll
    for (int c = 0; c < E; ++c) { acc[c] = make_float2(0.f, 0.f); nidx[c] = 0; }
    const int noct = (p.batch + T - 1) / T;
    for (int o = 0; o < noct; ++o) {
        const int b = o * T + t;
        const bool active = b < p.batch;
        const int bb = active ? b : 0;
        const float2* __restrict__ src = p.grid + (((int64_t)(bb / kIL) * p.k_outer + g0) * K) * kIL + (bb % kIL);
        const float2* __restrict__ csrc = p.coil + ((int64_t)bb * p.n_outer + n0) * N;
        int cnt = 0;
        auto ld = [&](int i) -> float2 { return active ? cconj(src[(int64_t)i * kIL]) : make_float2(0.f, 0.f); };
        auto st = [&](int i, float2 v) {
            const int n = (i + N / 2) & (K - 1);
            float2 r = cscale(cconj(v), so * __ldg(&sl[n]));
            r = active ? cmul(r, cconj(__ldg(&csrc[n]))) : make_float2(0.f, 0.f);
#pragma unroll
            for (int off = T / 2; off > 0; off >>= 1) {
                r.x += __shfl_xor_sync(0xffffffffu, r.x, off);
                r.y += __shfl_xor_sync(0xffffffffu, r.y, off);
            }
            acc[cnt] = cadd(acc[cnt], r);
            nidx[cnt] = n;
            ++cnt;
        };
        fft_line<K, false, true>(q0, true, lay, p.tw, ld, st);
        __syncthreads();          // the exchange buffers are reused by the next octet
    }
    if (t == 0) {
        float2* __restrict__ dst = p.img_out + (int64_t)n0 * N;
#pragma unroll
        for (int c = 0; c < E / 2; ++c) dst[nidx[c]] = acc[c];
    }
}

// ------------------------------------------------------------------------------------------------------------
// plan data of the interleaved path (built by plan_build_il in nufft.cu).  Two sample orders:
//   V order    key (column band, row k0_0, column):  kpack, delta, v2h
//   V^H order  key (column band, class, row k0_0, column), class 0 = column offset in the band >= 3 (the stencil
//              reaches into the next band), class 1 = the rest:  wtab, rowptr, pos, and every y_il array
// ------------------------------------------------------------------------------------------------------------
struct IlPlan {
    const uint32_t* kpack;    // V order: stencil base index per axis (10 bits each)
    const float* delta;       // V order: [2][M]
    const uint32_t* kpack_c;  // caller order (trajectory-coherent plans only, else null)
    const float* delta_c;     // caller order [2][M]
    const uint32_t* gbase;    // V order: base cell (row | col << 10) of the sample's window group (interp_il_win_kernel)
    const uint32_t* gbase_c;  // caller order (trajectory-coherent plans only, else null)
    const float* wv;          // coef_mode = 1: zero-padded weights [M][24] (w0 padded[10], 2 pad, w1 padded[10], 2 pad) in V order, else null
    const float* wv_c;        // ... in the caller's order
    const int32_t* v2h;       // V-order position -> V^H-order position
    const uint32_t* kpack_t;  // TILE order (interp_il_tile_kernel): stencil base index per axis
    const float* delta_t;     // tile order [2][M]
    const uint32_t* gbase_t;  // tile order: base of the sample's 8 x 8 window relative to the tile origin (row | col << 5)
    const float* wv_t;        // coef_mode = 1: weights [M][12] (w0[6], w1[6]) in tile order, else null
    const int32_t* t2h;       // tile-order position -> V^H-order position
    const int32_t* pos;       // caller's sample index -> V^H-order position
    const float* wtab;        // V^H order: [M][kTabW] = w0 rotated by the base row (slot (k0_0 + j) & 7 = w0[j], others 0), w1 part A[8], w1 part B[8] (float64-built)
    const int32_t* rowptr;    // [(band * 2 + class) * K0 + row]: first V^H-order sample of (band, class, row); + 1 entry
};

// a3: y = V grid.  One warp = 32 consecutive sorted samples x the 32 images of group blockIdx.y.
// Each lane prepares the weights of one sample (kb_weights) and stages them in shared memory; the warp then walks
// the samples one by one with warp-uniform weights: 36 loads of 256 contiguous bytes and 72 + 12 FMAs per lane.
constexpr int kInterpWarps = 8;
constexpr int kInterpChunk = 64;     // consecutive sorted samples per CTA
constexpr int kInterpChunkCaller = 64;   // ... in the caller-order variant (its output tile lives in shared memory)
// CALLER = false: samples are walked in V order and the output is y_il[group][V^H position][32] (coalesced rows);
//                 y_from_il_kernel restores the caller's order when needed.
// CALLER = true:  trajectory-coherent plans (consecutive caller samples are neighbours in k-space: radial spokes, spiral
//                 arms): samples are walked in the CALLER's order (kpack_c / delta_c), which has the same L1 locality
//                 along the readout, and the 64 x 32 result tile is written through shared memory straight into
//                 y[batch][M] (512 contiguous bytes per image): no layout pass at all.
template <bool CALLER, int CHUNK>
__global__ void __launch_bounds__(256)
interp_il_kernel(IlPlan s, GridGeom g, const float2* __restrict__ grid_il, float2* __restrict__ y_il, int batch,
                 KernelPoly P) {
    __shared__ float4 wrec[CHUNK * 4];
    __shared__ float2 otile[CALLER ? CHUNK : 1][33];
    const uint32_t* __restrict__ kpk = CALLER ? s.kpack_c : s.kpack;
    const float* __restrict__ dlt = CALLER ? s.delta_c : s.delta;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = blockIdx.y;
    const int64_t s0 = (int64_t)blockIdx.x * CHUNK;
    const int cnt = (int)min((int64_t)CHUNK, g.M - s0);
    for (int t = threadIdx.x; t < cnt; t += blockDim.x) {
        const int64_t si = s0 + t;
        const uint32_t kp = __ldg(&kpk[si]);
        float w0[kJ], w1[kJ];
        kb_weights(P, 0, __ldg(&dlt[si]), w0);
        kb_weights(P, 1, __ldg(&dlt[g.M + si]), w1);
        float4* r = &wrec[t * 4];
        r[0] = make_float4(w0[0], w0[1], w0[2], w0[3]);
        r[1] = make_float4(w0[4], w0[5], w1[0], w1[1]);
        r[2] = make_float4(w1[2], w1[3], w1[4], w1[5]);
        r[3] = make_float4(__int_as_float((int)(kp & 1023u)), __int_as_float((int)((kp >> 10) & 1023u)),
                           __int_as_float(CALLER ? 0 : __ldg(&s.v2h[si])), 0.f);
    }
    __syncthreads();
    const int K0 = g.K[0], K1 = g.K[1];
    const float2* __restrict__ G = grid_il + (int64_t)grp * g.cells * kIL + lane;
    // the warps of a CTA interleave over consecutive sorted samples: their stencils overlap, so the CTA's working set in
    // L1 is one moving window of a few rows instead of one window per warp
    for (int sidx = warp; sidx < cnt; sidx += kInterpWarps) {
        const float4 ra = wrec[sidx * 4 + 0], rb = wrec[sidx * 4 + 1];
        const float4 rc = wrec[sidx * 4 + 2], rd = wrec[sidx * 4 + 3];
        const float w0[kJ] = {ra.x, ra.y, ra.z, ra.w, rb.x, rb.y};
        const float w1[kJ] = {rb.z, rb.w, rc.x, rc.y, rc.z, rc.w};
        const int r0 = __float_as_int(rd.x), c0 = __float_as_int(rd.y);
        float2 acc = make_float2(0.f, 0.f);
        if (c0 + kJ <= K1) {
#pragma unroll
            for (int j0 = 0; j0 < kJ; ++j0) {
                const float2* __restrict__ pr = G + ((int64_t)((r0 + j0) & (K0 - 1)) * K1 + c0) * kIL;
                float2 r = make_float2(0.f, 0.f);
#pragma unroll
                for (int j1 = 0; j1 < kJ; ++j1) {
                    const float2 v = __ldg(pr + j1 * kIL);
                    r.x = fmaf(w1[j1], v.x, r.x);
                    r.y = fmaf(w1[j1], v.y, r.y);
                }
                acc.x = fmaf(w0[j0], r.x, acc.x);
                acc.y = fmaf(w0[j0], r.y, acc.y);
            }
        } else {      // stencil crosses the periodic seam of axis 1
#pragma unroll
            for (int j0 = 0; j0 < kJ; ++j0) {
                const float2* __restrict__ pr = G + (int64_t)((r0 + j0) & (K0 - 1)) * K1 * kIL;
                float2 r = make_float2(0.f, 0.f);
#pragma unroll
                for (int j1 = 0; j1 < kJ; ++j1) {
                    const float2 v = __ldg(pr + (int64_t)((c0 + j1) & (K1 - 1)) * kIL);
                    r.x = fmaf(w1[j1], v.x, r.x);
                    r.y = fmaf(w1[j1], v.y, r.y);
                }
                acc.x = fmaf(w0[j0], r.x, acc.x);
                acc.y = fmaf(w0[j0], r.y, acc.y);
            }
        }
        if (CALLER) otile[sidx][lane] = acc;
        else y_il[((int64_t)grp * g.M + __float_as_int(rd.z)) * kIL + lane] = acc;
    }
    if (CALLER) {     // y_il is the caller's y[batch][M] here: warp w writes images 4w .. 4w+3, 64 consecutive samples each
        __syncthreads();
#pragma unroll
        for (int li = 0; li < kIL / kInterpWarps; ++li) {
            const int l = warp * (kIL / kInterpWarps) + li, b = grp * kIL + l;
            if (b >= batch) continue;
            for (int t = lane; t < cnt; t += 32) y_il[(int64_t)b * g.M + s0 + t] = otile[t][l];
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// a3 with register windows (round 2).  profiles/r01n: interp_il_kernel re-reads all 36 stencil cells of every sample
// (36 warp loads of 256 B = 72 L1 wavefronts per sample and image group) and sits on the L1 data pipe (85 % busy) at 26 %
// of the HBM roofline.  Neighbouring samples of the walk order (one grid cell apart along a radial readout; many per cell
// near the k-space centre) share most of their stencils, so the plan cuts the walk order into GROUPS -- maximal runs of
// consecutive samples whose stencil bases fit a 3 x 3 box -- and a warp keeps the 8 x 8 cells x 32 images WINDOW of the
// current group in registers (128 registers per lane): 64 loads per group instead of 36 per sample (config 2: 3.2 samples
// per group in the caller's order, 5.2 in the sorted order).  Per sample the lane then runs 72 packed FMAs (FFMA2 on
// (re, im), scalar weights) with weights that are zero outside the sample's own 6 x 6 support: the arithmetic is that of
// the plain stencil sum.  Weights are evaluated once per sample by one lane (kb_weights) and parked zero-padded in shared
// memory; all per-sample loads are warp-uniform broadcasts.
// ------------------------------------------------------------------------------------------------------------
constexpr int kIwWarps = 4;          // warps per CTA, 32 consecutive samples of the walk order each
constexpr int kIwRec = 28;           // floats per staged sample: w0 padded [10], 2 pad, w1 padded [10], 2 pad, key, output index, 2 pad
                                     // (7 float4: 7 s mod 8 is a permutation -> conflict-free 128-bit stores)
// Window shapes (rows x columns of grid cells, <= 64 cells = 128 registers per lane).  A readout that runs along the grid
// columns stays in ONE stencil base row for many samples: a 6 x 10 window then serves five samples where the 8 x 8 one
// serves three.  The plan picks, group by group, the shape with the fewest window cells per sample (config 2, caller's
// order: 20.1 cells per sample with 8 x 8 alone, 15.9 with the five shapes).  shape id -> (rows, columns):
constexpr int kIwShapes = 5;
__host__ __device__ __forceinline__ constexpr int iw_rows(int sh) { return sh == 0 ? 8 : (sh == 1 ? 6 : (sh == 2 ? 10 : (sh == 3 ? 7 : 9))); }
__host__ __device__ __forceinline__ constexpr int iw_cols(int sh) { return sh == 0 ? 8 : (sh == 1 ? 10 : (sh == 2 ? 6 : (sh == 3 ? 9 : 7))); }
// group key (plan, per sample): base row | base column << 10 | shape << 20

// zero-padded weight vector of up to 10 entries: p[i] = w[i - o], 0 <= i - o < 6, else 0   (o in 0..4)
__device__ __forceinline__ void il_pad10(const float (&w)[kJ], int o, float (&p)[12]) {
#pragma unroll
    for (int i = 0; i < 12; ++i) {
        float v = 0.f;
#pragma unroll
        for (int oo = 0; oo < 5; ++oo)
            if (i - oo >= 0 && i - oo < kJ) v = (o == oo) ? w[i - oo] : v;
        p[i] = v;
    }
}

// one group of the walk: load its R x C window once, then interpolate its samples t, t + 1, ... while the key stays the same
template <int R, int C, bool CALLER>
__device__ __forceinline__ int iw_group(const float* __restrict__ recw, int t, int cnt, int key, const float2* __restrict__ G,
                                        int K0, int K1, float2 (*otile)[33], int obase, float2* __restrict__ y_il_grp, int lane) {
    float2 win[R][C];
    const int br = key & 1023, bc = (key >> 10) & 1023;
    if (bc + C <= K1) {
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const float2* __restrict__ pr = G + ((int64_t)((br + i) & (K0 - 1)) * K1 + bc) * kIL;
#pragma unroll
            for (int j = 0; j < C; ++j) win[i][j] = __ldg(pr + j * kIL);
        }
    } else {      // the window crosses the periodic seam of axis 1
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const float2* __restrict__ pr = G + (int64_t)((br + i) & (K0 - 1)) * K1 * kIL;
#pragma unroll
            for (int j = 0; j < C; ++j) win[i][j] = __ldg(pr + (int64_t)((bc + j) & (K1 - 1)) * kIL);
        }
    }
    do {
        const float* r = recw + t * kIwRec;
        float w0[12], w1[12];
#pragma unroll
        for (int v4 = 0; v4 < 3; ++v4) {
            const float4 a = *reinterpret_cast<const float4*>(r + 4 * v4), b = *reinterpret_cast<const float4*>(r + 12 + 4 * v4);
            w0[4 * v4] = a.x; w0[4 * v4 + 1] = a.y; w0[4 * v4 + 2] = a.z; w0[4 * v4 + 3] = a.w;
            w1[4 * v4] = b.x; w1[4 * v4 + 1] = b.y; w1[4 * v4 + 2] = b.z; w1[4 * v4 + 3] = b.w;
        }
        float2 acc = make_float2(0.f, 0.f);
#pragma unroll
        for (int i = 0; i < R; ++i) {
            float2 rs = __fmul2_rn(make_float2(w1[0], w1[0]), win[i][0]);
#pragma unroll
            for (int j = 1; j < C; ++j) rs = __ffma2_rn(make_float2(w1[j], w1[j]), win[i][j], rs);
            acc = __ffma2_rn(make_float2(w0[i], w0[i]), rs, acc);
        }
        if (CALLER) otile[obase + t][lane] = acc;
        else y_il_grp[(int64_t)__float_as_int(r[25]) * kIL + lane] = acc;
        ++t;
    } while (t < cnt && __float_as_int(recw[t * kIwRec + 24]) == key);
    return t;
}

template <bool CALLER>
__global__ void __launch_bounds__(kIwWarps * 32, 3)
interp_il_win_kernel(IlPlan s, GridGeom g, const float2* __restrict__ grid_il, float2* __restrict__ y_out, int batch,
                     KernelPoly P) {
    pdl_enter();
    __shared__ __align__(16) float recs[kIwWarps][32][kIwRec];
    __shared__ float2 otile[CALLER ? kIwWarps * 32 : 1][33];
    const uint32_t* __restrict__ kpk = CALLER ? s.kpack_c : s.kpack;
    const float* __restrict__ dlt = CALLER ? s.delta_c : s.delta;
    const uint32_t* __restrict__ gbs = CALLER ? s.gbase_c : s.gbase;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = blockIdx.y;
    const int64_t s0 = (int64_t)blockIdx.x * (kIwWarps * 32);
    const int K0 = g.K[0], K1 = g.K[1];
    const float2* __restrict__ G = grid_il + (int64_t)grp * g.cells * kIL + lane;
    const int64_t w0s = s0 + warp * 32;
    const int cnt = (int)max((int64_t)0, min((int64_t)32, g.M - w0s));
    if (lane < cnt) {   // stage: lane = sample
        const int64_t si = w0s + lane;
        const uint32_t gb = __ldg(&gbs[si]);
        float* r = &recs[warp][lane][0];
        const float* __restrict__ wt = CALLER ? s.wv_c : s.wv;
        if (wt) {       // coef_mode = 1: precomputed (float64-built) padded weights, 96 contiguous bytes per sample
            const float4* __restrict__ t4 = reinterpret_cast<const float4*>(wt + si * 24);
#pragma unroll
            for (int v4 = 0; v4 < 6; ++v4) reinterpret_cast<float4*>(r)[v4] = __ldg(t4 + v4);
        } else {
            const uint32_t kp = __ldg(&kpk[si]);
            float w[kJ], pd[12];
            kb_weights(P, 0, __ldg(&dlt[si]), w);
            il_pad10(w, (int)(kp & 1023u) - (int)(gb & 1023u), pd);
#pragma unroll
            for (int v4 = 0; v4 < 3; ++v4) reinterpret_cast<float4*>(r)[v4] = make_float4(pd[4 * v4], pd[4 * v4 + 1], pd[4 * v4 + 2], pd[4 * v4 + 3]);
            kb_weights(P, 1, __ldg(&dlt[g.M + si]), w);
            il_pad10(w, (int)((kp >> 10) & 1023u) - (int)((gb >> 10) & 1023u), pd);
#pragma unroll
            for (int v4 = 0; v4 < 3; ++v4) reinterpret_cast<float4*>(r)[3 + v4] = make_float4(pd[4 * v4], pd[4 * v4 + 1], pd[4 * v4 + 2], pd[4 * v4 + 3]);
        }
        reinterpret_cast<float4*>(r)[6] = make_float4(__int_as_float((int)gb), __int_as_float(CALLER ? 0 : __ldg(&s.v2h[si])), 0.f, 0.f);
    }
    __syncwarp();
    const float* recw = &recs[warp][0][0];
    float2* __restrict__ yg = CALLER ? nullptr : y_out + (int64_t)grp * g.M * kIL;
    int t = 0;
#pragma unroll 1
    while (t < cnt) {
        const int key = __float_as_int(recw[t * kIwRec + 24]);
        switch ((key >> 20) & 7) {       // warp-uniform
            case 1: t = iw_group<iw_rows(1), iw_cols(1), CALLER>(recw, t, cnt, key, G, K0, K1, otile, warp * 32, yg, lane); break;
            case 2: t = iw_group<iw_rows(2), iw_cols(2), CALLER>(recw, t, cnt, key, G, K0, K1, otile, warp * 32, yg, lane); break;
            case 3: t = iw_group<iw_rows(3), iw_cols(3), CALLER>(recw, t, cnt, key, G, K0, K1, otile, warp * 32, yg, lane); break;
            case 4: t = iw_group<iw_rows(4), iw_cols(4), CALLER>(recw, t, cnt, key, G, K0, K1, otile, warp * 32, yg, lane); break;
            default: t = iw_group<iw_rows(0), iw_cols(0), CALLER>(recw, t, cnt, key, G, K0, K1, otile, warp * 32, yg, lane); break;
        }
    }
    if (CALLER) {     // y_out is the caller's y[batch][M]: warp w writes images 8 w .. 8 w + 7, 128 consecutive samples each
        __syncthreads();
        const int tot = (int)min((int64_t)(kIwWarps * 32), g.M - s0);
#pragma unroll
        for (int li = 0; li < kIL / kIwWarps; ++li) {
            const int l = warp * (kIL / kIwWarps) + li, b = grp * kIL + l;
            if (b >= batch) continue;
            for (int tt = lane; tt < tot; tt += 32) y_out[(int64_t)b * g.M + s0 + tt] = otile[tt][l];
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// a3 with register windows fed from a SHARED tile (round 2, the sorted walk of A^H A and of the incoherent trajectories).
// profiles/r02a: interp_il_win_kernel loads every window from L2 (16 KB per group and warp, L1 hit rate 3 %) and sits at
// ~10 TB/s of L2 -> SM traffic.  Here the CTA = one work item (tile of T x T stencil base cells, <= NW * 32 of its samples)
// x one image group: the padded (T+5)^2 cells x 32 images tile is staged ONCE by the copy engine (one tensor-map copy, SASS
// UTMALDG; tiles on the periodic seam: one bulk copy per row segment) while the warps evaluate their samples' weights;
// the windows of the groups are then read from shared memory (conflict-free 256-B rows): L2 -> SM traffic is
// ((T+5)/T)^2 x the grid instead of 11 cells per sample.  Two CTAs per SM: one loads while the other computes.
// Every sample jumps, warp-uniformly, to the code variant of its support offset inside the window: exactly 36 + 6 packed
// FMAs per sample instead of the 72 zero-padded ones of interp_il_win_kernel (measured: the padded form is FMA-pipe bound
// here once the loads come from shared memory).  Output rows y_il[group][V^H position][32].
// Plan data in TILE order (IlPlan::kpack_t ...): samples sorted by tile, inside a tile by 3 x 3 blocks of base cells; a warp
// takes a contiguous share of the item; group key = base of the group's 8 x 8 window relative to the tile origin (row | col << 5).
// ------------------------------------------------------------------------------------------------------------
constexpr int kItRec = 20;           // floats per staged sample: w0[6], w1[6], group key, output row, variant, pad (80 B: conflict-free 128-bit stores)
template <int T, int NW> struct IlTile {
    static constexpr int PW = T + kJ - 1;                       // padded tile edge in cells
    static constexpr int TILE_BYTES = PW * PW * kIL * 8;
    static constexpr int REC_BYTES = NW * 32 * kItRec * 4;
    static constexpr int SMEM = TILE_BYTES + REC_BYTES + 16;
    static constexpr int CAP = NW * 32;                         // samples per work item
};
constexpr int kItT = 14;             // stencil base cells per tile and axis: padded tile 19 x 19 cells x 32 images = 92 KB
constexpr int kItWarps = 6;          // warps per CTA (two CTAs per SM)
constexpr int kItWin = 8;            // window edge in cells (8 x 8 cells = 128 registers per lane)
constexpr int kItAhead = 160;        // plan data of the item this many items later is prefetched into L2
struct IlTileItem { int32_t start; int32_t cnt; int32_t r0; int32_t c0; };    // tile-order sample range, tile origin (cells)

// the 6 x 6 stencil of a sample whose support starts at (O0, O1) inside the R x C register window
template <int R, int C, int O0, int O1>
__device__ __forceinline__ float2 it_eval(const float2 (&win)[R][C], const float (&w0)[kJ], const float (&w1)[kJ]) {
    float2 acc0 = make_float2(0.f, 0.f), acc1 = make_float2(0.f, 0.f);
#pragma unroll
    for (int i = 0; i < kJ; ++i) {
        float2 rs = __fmul2_rn(make_float2(w1[0], w1[0]), win[O0 + i][O1]);
#pragma unroll
        for (int j = 1; j < kJ; ++j) rs = __ffma2_rn(make_float2(w1[j], w1[j]), win[O0 + i][O1 + j], rs);
        if (i & 1) acc1 = __ffma2_rn(make_float2(w0[i], w0[i]), rs, acc1);
        else acc0 = __ffma2_rn(make_float2(w0[i], w0[i]), rs, acc0);
    }
    return __fadd2_rn(acc0, acc1);
}
#define NU_IT_VARIANT(V)                                                                     \
    case V:                                                                                  \
        if constexpr (V < (R - kJ + 1) * (C - kJ + 1))                                        \
            acc = it_eval<R, C, V / (C - kJ + 1), V % (C - kJ + 1)>(win, w0, w1);             \
        break;

// one group of the walk: load its R x C window from the shared tile once, then interpolate its samples t, t + 1, ... while
// the key stays the same
template <int R, int C, int PW>
__device__ __forceinline__ int it_group(const float* __restrict__ recw, int t, int cnt, int key, const float2* __restrict__ tl,
                                        float2* __restrict__ y_il_grp, int lane) {
    float2 win[R][C];
    const float2* __restrict__ base = tl + ((key & 31) * PW + ((key >> 5) & 31)) * kIL;
#pragma unroll
    for (int i = 0; i < R; ++i)
#pragma unroll
        for (int j = 0; j < C; ++j) win[i][j] = base[(i * PW + j) * kIL];
    do {
        const float4* r4 = reinterpret_cast<const float4*>(recw + t * kItRec);
        const float4 a = r4[0], b = r4[1], c = r4[2], d = r4[3];
        const float w0[kJ] = {a.x, a.y, a.z, a.w, b.x, b.y};
        const float w1[kJ] = {b.z, b.w, c.x, c.y, c.z, c.w};
        float2 acc = make_float2(0.f, 0.f);
        switch (__float_as_int(d.z)) {       // warp-uniform
            NU_IT_VARIANT(0) NU_IT_VARIANT(1) NU_IT_VARIANT(2) NU_IT_VARIANT(3) NU_IT_VARIANT(4)
            NU_IT_VARIANT(5) NU_IT_VARIANT(6) NU_IT_VARIANT(7) NU_IT_VARIANT(8)
            default: break;
        }
        y_il_grp[(int64_t)__float_as_int(d.y) * kIL + lane] = acc;
        ++t;
    } while (t < cnt && __float_as_int(recw[t * kItRec + 12]) == key);
    return t;
}

template <int T, int NW, int MB>
__global__ void __launch_bounds__(NW * 32, MB)
interp_il_tile_kernel(IlPlan s, GridGeom g, const IlTileItem* __restrict__ items, int n_items, int ngroups,
                      const float2* __restrict__ grid_il, float2* __restrict__ y_il, KernelPoly P,
                      const __grid_constant__ CUtensorMap tmap, int use_tmap) {
    using G = IlTile<T, NW>;
    constexpr int PW = G::PW;
    extern __shared__ __align__(128) unsigned char it_smem[];
    float2* tile = reinterpret_cast<float2*>(it_smem);                              // [PW][PW][32]
    float* recs = reinterpret_cast<float*>(it_smem + G::TILE_BYTES);                // [NW][32][kItRec]
    uint64_t* bar = reinterpret_cast<uint64_t*>(it_smem + G::TILE_BYTES + G::REC_BYTES);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // the image groups of one item run next to each other: the second one finds the item's plan data in L2
    const int grp = blockIdx.x % ngroups, item = blockIdx.x / ngroups;
    const IlTileItem it = items[item];
    const int K0 = g.K[0], K1 = g.K[1];
    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    // plan data of the item that starts kItAhead items later is pulled into L2 now (it comes from DRAM otherwise: two
    // dependent misses at the head of every CTA)
    IlTileItem nxt{0, 0, 0, 0};
    const bool pf = warp == NW - 1 && grp == 0 && item + kItAhead < n_items;
    if (pf) nxt = items[item + kItAhead];
    pdl_enter();      // the grid is the previous kernel's output
    if (warp == 0) {
        const bool inside = it.r0 + PW <= K0 && it.c0 + PW <= K1;
        if (use_tmap && inside) {
            if (lane == 0) {
                mbar_expect_tx(bar, (uint32_t)G::TILE_BYTES);
                tma_load_tile_4d(tile, &tmap, 0, it.c0, it.r0, grp, bar);
            }
        } else {
            if (lane == 0) mbar_expect_tx(bar, (uint32_t)G::TILE_BYTES);
            __syncwarp();
            const float2* __restrict__ Gg = grid_il + (int64_t)grp * g.cells * kIL;
            if (lane < PW) {      // one padded row per lane, split where it crosses the seam of axis 1
                const float2* __restrict__ row = Gg + (int64_t)((it.r0 + lane) & (K0 - 1)) * K1 * kIL;
                const int n1 = min(PW, K1 - it.c0);
                bulk_g2s(tile + (lane * PW) * kIL, row + (int64_t)it.c0 * kIL, (uint32_t)(n1 * kIL * 8), bar);
                if (n1 < PW) bulk_g2s(tile + (lane * PW + n1) * kIL, row, (uint32_t)((PW - n1) * kIL * 8), bar);
            }
        }
    }
    // the warp's share of the item; lane = sample while staging
    const int per = (it.cnt + NW - 1) / NW;
    const int t0 = warp * per;
    const int cnt = max(0, min(per, it.cnt - t0));
    float* recw = recs + warp * 32 * kItRec;
    if (lane < cnt) {
        const int64_t si = (int64_t)it.start + t0 + lane;
        const uint32_t gb = __ldg(&s.gbase_t[si]);
        const uint32_t kp = __ldg(&s.kpack_t[si]);
        const int32_t orow = __ldg(&s.t2h[si]);
        float w0[kJ], w1[kJ];
        if (s.wv_t) {       // coef_mode = 1: precomputed (float64-built) weights, 48 contiguous bytes per sample
            const float4* __restrict__ t4 = reinterpret_cast<const float4*>(s.wv_t + si * 12);
            const float4 a = __ldg(t4), b = __ldg(t4 + 1), c = __ldg(t4 + 2);
            w0[0] = a.x; w0[1] = a.y; w0[2] = a.z; w0[3] = a.w; w0[4] = b.x; w0[5] = b.y;
            w1[0] = b.z; w1[1] = b.w; w1[2] = c.x; w1[3] = c.y; w1[4] = c.z; w1[5] = c.w;
        } else {
            kb_weights(P, 0, __ldg(&s.delta_t[si]), w0);
            kb_weights(P, 1, __ldg(&s.delta_t[g.M + si]), w1);
        }
        const int o0 = (int)(kp & 1023u) - it.r0 - (int)(gb & 31u), o1 = (int)((kp >> 10) & 1023u) - it.c0 - (int)((gb >> 5) & 31u);
        float4* r4 = reinterpret_cast<float4*>(recw + lane * kItRec);
        r4[0] = make_float4(w0[0], w0[1], w0[2], w0[3]);
        r4[1] = make_float4(w0[4], w0[5], w1[0], w1[1]);
        r4[2] = make_float4(w1[2], w1[3], w1[4], w1[5]);
        r4[3] = make_float4(__int_as_float((int)gb), __int_as_float(orow), __int_as_float(o0 * (kItWin - kJ + 1) + o1), 0.f);
    }
    if (pf) {         // 5 arrays x (<= NW * 32 entries x 4 B), one 128-B line per lane and round
        constexpr int LPA = (NW * 32 * 4 + 127) / 128 + 1;      // lines per array (+1: the range is not line-aligned)
        for (int q = lane; q < 5 * LPA; q += 32) {
            const int arr = q / LPA, ln = q % LPA;
            const char* bp = arr == 0 ? (const char*)(s.gbase_t + nxt.start) : arr == 1 ? (const char*)(s.kpack_t + nxt.start)
                           : arr == 2 ? (const char*)(s.t2h + nxt.start) : arr == 3 ? (const char*)(s.delta_t + nxt.start)
                           : (const char*)(s.delta_t + g.M + nxt.start);
            if (ln * 128 < nxt.cnt * 4 + 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(bp + ln * 128));
        }
    }
    __syncwarp();
    mbar_wait(bar, 0);
    const float2* __restrict__ tl = tile + lane;
    float2* __restrict__ yg = y_il + (int64_t)grp * g.M * kIL;
    int t = 0;
#pragma unroll 1
    while (t < cnt) {
        const int key = __float_as_int(recw[t * kItRec + 12]);
        t = it_group<kItWin, kItWin, PW>(recw, t, cnt, key, tl, yg, lane);
    }
}

// Layout changes of the sample vectors, coalesced on both sides (a warp moves a 32 samples x 32 images tile through
// shared memory): the caller's y[batch][M] <-> y_il[group][sorted position][32].  pos[m] = sorted position of caller
// sample m.  Idle lanes of the last group are written as zeros.
__global__ void __launch_bounds__(128)
y_to_il_kernel(const int32_t* __restrict__ pos, const float2* __restrict__ y, float2* __restrict__ y_il, int64_t M,
               int batch) {
    pdl_enter();
    __shared__ float2 tile[4][32][33];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = blockIdx.y;
    const int64_t m0 = ((int64_t)blockIdx.x * 4 + warp) * 32;
    if (m0 >= M) return;
    const int cnt = (int)min((int64_t)32, M - m0);
    const int my = (lane < cnt) ? __ldg(&pos[m0 + lane]) : 0;
    // all 32 row loads of the warp are issued before the first one is consumed (the pass is latency-bound otherwise)
    float2 v[kIL];
#pragma unroll
    for (int l = 0; l < kIL; ++l) {
        const int b = grp * kIL + l;
        v[l] = (lane < cnt && b < batch) ? __ldg(&y[(int64_t)b * M + m0 + lane]) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int l = 0; l < kIL; ++l) tile[warp][lane][l] = v[l];
    __syncwarp();
    float2* __restrict__ dst = y_il + (int64_t)grp * M * kIL + lane;
    for (int k = 0; k < cnt; ++k) {
        const int i = __shfl_sync(0xffffffffu, my, k);
        dst[(int64_t)i * kIL] = tile[warp][k][lane];
    }
}

__global__ void __launch_bounds__(128)
y_from_il_kernel(const int32_t* __restrict__ pos, const float2* __restrict__ y_il, float2* __restrict__ y, int64_t M,
                 int batch) {
    pdl_enter();
    __shared__ float2 tile[4][32][33];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = blockIdx.y;
    const int64_t m0 = ((int64_t)blockIdx.x * 4 + warp) * 32;
    if (m0 >= M) return;
    const int cnt = (int)min((int64_t)32, M - m0);
    const int my = (lane < cnt) ? __ldg(&pos[m0 + lane]) : 0;
    const float2* __restrict__ src = y_il + (int64_t)grp * M * kIL + lane;
    // all 32 row loads are issued before the first one is consumed (as in y_to_il_kernel: the pass is latency-bound otherwise)
    float2 v[kIL];
#pragma unroll
    for (int k = 0; k < kIL; ++k) {
        const int i = __shfl_sync(0xffffffffu, my, k);
        v[k] = (k < cnt) ? __ldg(&src[(int64_t)i * kIL]) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int k = 0; k < kIL; ++k) tile[warp][k][lane] = v[k];
    __syncwarp();
    if (lane >= cnt) return;
#pragma unroll 8
    for (int l = 0; l < kIL; ++l) {
        const int b = grp * kIL + l;
        if (b < batch) y[(int64_t)b * M + m0 + lane] = tile[warp][lane][l];
    }
}

// ------------------------------------------------------------------------------------------------------------
// a4: grid = V^H y, gather form with register accumulators (see the header of this file)
// ------------------------------------------------------------------------------------------------------------
struct IlItem {
    int32_t cb;       // column band: grid columns 8 cb .. 8 cb + 7
    int32_t r0;       // first grid row of the item
    int32_t nrows;    // 8, 4, 2 or 1 rows; the 8 warps of the CTA split each row's sample list 8 / nrows ways
    int32_t load;     // row-sample interactions of the item (plan-time cost estimate; sort key)
};

constexpr int kStageCap = 48;      // samples per list per staging round (one group per CTA)
constexpr int kStageCap2 = 40;     // ... when a CTA handles two groups (64 images)
template <int NG> struct GridStage {
    static constexpr int CAP = (NG == 1) ? kStageCap : kStageCap2;
    static constexpr int BYTES = 3 * CAP * (kTabW * 4 + NG * kIL * 8) + 16;
};

// Adds staged samples [i0, i1) (indices into one staged list) to the accumulators of output row `row`, for NG groups of
// 32 images that share the staged table records (weights, row lookup): only the y row and the FMAs are per group.
// Accumulators are kept as packed pairs for Blackwell's two-wide FP32 FMA (fma.rn.f32x2, SASS FFMA2):
// ax[k] = (re of cell 2k, re of cell 2k+1), ay[k] = the imaginary parts; the weight pair of two adjacent cells is one
// aligned register pair straight out of the 128-bit table load, so one FFMA2 updates two cells.
template <int OFF, int NG, int CAP>
__device__ __forceinline__ void il_accumulate_smem(float2 (&ax)[NG][kBandW / 2], float2 (&ay)[NG][kBandW / 2],
                                                   const float* __restrict__ rec_s, const float2* __restrict__ y_s,
                                                   int row, int i0, int i1) {
#pragma unroll 4
    for (int i = i0; i < i1; ++i) {
        const float* rec = rec_s + i * kTabW;
        const float w0 = rec[row & 7];        // w0 is stored rotated by the stencil base row (slot (k0_0 + j) & 7 = w0[j])
        const float4 pa = *reinterpret_cast<const float4*>(rec + OFF);
        const float4 pb = *reinterpret_cast<const float4*>(rec + OFF + 4);
#pragma unroll
        for (int gq = 0; gq < NG; ++gq) {
            const float2 yv = y_s[(gq * 3 * CAP + i) * kIL];
            const float tx = w0 * yv.x, ty = w0 * yv.y;
            const float2 txx = make_float2(tx, tx), tyy = make_float2(ty, ty);
            ax[gq][0] = __ffma2_rn(make_float2(pa.x, pa.y), txx, ax[gq][0]); ay[gq][0] = __ffma2_rn(make_float2(pa.x, pa.y), tyy, ay[gq][0]);
            ax[gq][1] = __ffma2_rn(make_float2(pa.z, pa.w), txx, ax[gq][1]); ay[gq][1] = __ffma2_rn(make_float2(pa.z, pa.w), tyy, ay[gq][1]);
            ax[gq][2] = __ffma2_rn(make_float2(pb.x, pb.y), txx, ax[gq][2]); ay[gq][2] = __ffma2_rn(make_float2(pb.x, pb.y), tyy, ay[gq][2]);
            ax[gq][3] = __ffma2_rn(make_float2(pb.z, pb.w), txx, ax[gq][3]); ay[gq][3] = __ffma2_rn(make_float2(pb.z, pb.w), tyy, ay[gq][3]);
        }
    }
}

// CTA = one work item (band, nrows rows) x NG groups of 32 images (blockIdx.y = first group / NG, plus group0).  The
// samples that touch the item's rows are, per list (this band class 0, this band class 1, previous band class 0), ONE
// contiguous range of the V^H order (two at the periodic row seam), so their table records (96 B each) and their y_il
// rows (256 B each per group) are contiguous in global memory: one elected thread issues bulk copies of up to CAP samples
// per list into shared memory, all warps wait on the mbarrier, and every warp then accumulates its own row from shared
// memory.  Global-memory latency is paid once per round per CTA instead of once per warp per four samples.
template <int NG>
__global__ void __launch_bounds__(256)
gridding_il_kernel(IlPlan s, GridGeom g, const IlItem* __restrict__ items, const float2* __restrict__ y_il,
                   float2* __restrict__ grid_il, int group0) {
    pdl_enter();
    constexpr int CAP = GridStage<NG>::CAP;
    extern __shared__ __align__(128) unsigned char gsm[];
    float2* y_s = reinterpret_cast<float2*>(gsm);                                           // [NG][3][CAP][32]
    float* rec_s = reinterpret_cast<float*>(gsm + NG * 3 * CAP * kIL * 8);                  // [3][CAP][24]
    uint64_t* bar = reinterpret_cast<uint64_t*>(gsm + 3 * CAP * (NG * kIL * 8 + kTabW * 4));
    const IlItem it = items[blockIdx.x];
    const int grp = group0 + blockIdx.y * NG;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nsplit = 8 / it.nrows, lsplit = 31 - __clz(nsplit);       // nsplit is a power of two
    const int row = it.r0 + (warp >> lsplit), part = warp & (nsplit - 1);
    const int K0 = g.K[0], K1 = g.K[1], nb = K1 / kBandW;
    const int cbp = (it.cb + nb - 1) % nb;
    const float2* __restrict__ Y = y_il + (int64_t)grp * g.M * kIL;
    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    uint32_t phase = 0;
    float2 ax[NG][kBandW / 2], ay[NG][kBandW / 2];
#pragma unroll
    for (int gq = 0; gq < NG; ++gq)
#pragma unroll
        for (int c = 0; c < kBandW / 2; ++c) { ax[gq][c] = make_float2(0.f, 0.f); ay[gq][c] = make_float2(0.f, 0.f); }
    // stencil base rows that touch the item: r0-5 .. r0+nrows-1 (mod K0): one row segment, or two at the seam
    const int nseg = (it.r0 >= kJ - 1) ? 1 : 2;
#pragma unroll 1
    for (int sg = 0; sg < nseg; ++sg) {
        const int slo = (sg == 0) ? max(it.r0 - (kJ - 1), 0) : K0 - (kJ - 1) + it.r0;
        const int shi = (sg == 0) ? it.r0 + it.nrows - 1 : K0 - 1;
        const int shift = (sg == 0) ? 0 : K0;
        int cbeg[3], cend[3], wbeg[3], wend[3];
        const int wlo = max(slo, row + shift - (kJ - 1)), whi = min(shi, row + shift);
        int rounds = 0;
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const int base = ((q == 2 ? cbp : it.cb) * 2 + (q == 1 ? 1 : 0)) * K0;
            cbeg[q] = __ldg(&s.rowptr[base + slo]);
            cend[q] = __ldg(&s.rowptr[base + shi + 1]);
            if (wlo <= whi) { wbeg[q] = __ldg(&s.rowptr[base + wlo]); wend[q] = __ldg(&s.rowptr[base + whi + 1]); }
            else { wbeg[q] = 0; wend[q] = 0; }
            rounds = max(rounds, (cend[q] - cbeg[q] + CAP - 1) / CAP);
        }
#pragma unroll 1
        for (int k = 0; k < rounds; ++k) {
            if (threadIdx.x == 0) {
                uint32_t bytes = 0;
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    const int c0 = cbeg[q] + k * CAP, n = min(CAP, cend[q] - c0);
                    if (n > 0) bytes += (uint32_t)n * (kTabW * 4 + NG * kIL * 8);
                }
                mbar_expect_tx(bar, bytes);
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    const int c0 = cbeg[q] + k * CAP, n = min(CAP, cend[q] - c0);
                    if (n > 0) {
                        bulk_g2s(rec_s + q * CAP * kTabW, s.wtab + (int64_t)c0 * kTabW, (uint32_t)n * kTabW * 4, bar);
#pragma unroll
                        for (int gq = 0; gq < NG; ++gq)
                            bulk_g2s(y_s + (gq * 3 + q) * CAP * kIL, Y + ((int64_t)gq * g.M + c0) * kIL,
                                     (uint32_t)n * kIL * 8, bar);
                    }
                }
            }
            mbar_wait(bar, phase);
            phase ^= 1;
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                const int c0 = cbeg[q] + k * CAP, c1 = min(c0 + CAP, cend[q]);
                const int x0 = max(wbeg[q], c0), x1 = min(wend[q], c1);       // my row's samples within the staged chunk
                if (x1 > x0) {
                    const int n = x1 - x0;
                    const int i0 = x0 - c0 + ((n * part) >> lsplit), i1 = x0 - c0 + ((n * (part + 1)) >> lsplit);
                    if (q == 2) il_accumulate_smem<16, NG, CAP>(ax, ay, rec_s + q * CAP * kTabW, y_s + q * CAP * kIL + lane, row, i0, i1);
                    else        il_accumulate_smem<8, NG, CAP>(ax, ay, rec_s + q * CAP * kTabW, y_s + q * CAP * kIL + lane, row, i0, i1);
                }
            }
            __syncthreads();      // every warp is done with the staged chunk before the next round overwrites it
        }
    }
#pragma unroll
    for (int gq = 0; gq < NG; ++gq) {
        float2 acc[kBandW];
#pragma unroll
        for (int c = 0; c < kBandW / 2; ++c) {
            acc[2 * c] = make_float2(ax[gq][c].x, ay[gq][c].x);
            acc[2 * c + 1] = make_float2(ax[gq][c].y, ay[gq][c].y);
        }
        if (nsplit > 1) {       // fixed-order sum of the partial accumulators of one row (staging area reused)
            float2* red = y_s;  // [8][kBandW][32]
            if (gq > 0) __syncthreads();
#pragma unroll
            for (int c = 0; c < kBandW; ++c) red[(warp * kBandW + c) * kIL + lane] = acc[c];
            __syncthreads();
            if (part == 0)
                for (int q = 1; q < nsplit; ++q)
#pragma unroll
                    for (int c = 0; c < kBandW; ++c) acc[c] = cadd(acc[c], red[((warp + q) * kBandW + c) * kIL + lane]);
        }
        if (part == 0) {
            float2* __restrict__ dst = grid_il + (((int64_t)(grp + gq) * K0 + row) * K1 + it.cb * kBandW) * kIL + lane;
#pragma unroll
            for (int c = 0; c < kBandW; ++c) dst[c * kIL] = acc[c];
        }
    }
}

// x[n] = sum_b img[b][n]  is done by coil_sum_kernel (solver.cuh).

}  // namespace nufft
