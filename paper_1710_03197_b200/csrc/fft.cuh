// fft.cuh -- hand-written shared-memory FFT kernel set of the NUFFT hot path (steps a1, a2, a5, a6 of
// SURVEY.md section 8(a)).  cuFFT is not used anywhere in the product.
//
// One K-point line is computed as a 2- or 3-stage Cooley-Tukey decomposition K = R1*R2*R3 with radices in {4,8,16}:
//   input index  n = n1*(K/R1) + n2*(K/(R1 R2)) + n3,     output index k = k1 + R1*k2 + R1*R2*k3.
// Stage s works on the data seen as (kA, n_s, nB): kA = output digits produced so far (range A), n_s the digit
// being transformed (range R), nB the remaining input digits (range B = K/(A R)).  After the radix-R butterfly the
// result is multiplied by W_K^{A nB k_s} and exchanged through shared memory.  Stage 1 reads global memory directly
// (coalesced: consecutive threads hold consecutive nB) and the last stage writes global memory directly (consecutive
// threads hold consecutive kA), so the line crosses shared memory only between stages.
//
// Fusions:  a1 scaling + circular zero-pad live in the stage-1 loader of the first pass;  the padded
// half of every input line is known to be zero and is neither loaded nor stored anywhere (input pruning);  the
// adjoint passes compute only the N of K outputs that survive the crop (output pruning) and the last one applies
// S^H.  The inverse transform is conj(FFT(conj(.))), the conjugations folded into loader / storer.
#pragma once
#include "common.cuh"

namespace nufft {

// ------------------------------------------------------------------------------------------------------------
// radix butterflies: in-place forward DFT (e^{-2 pi i nk/R}) of R values, natural order in and out
// ------------------------------------------------------------------------------------------------------------
template <int R> struct Bfly;

template <> struct Bfly<2> {
    static __device__ __forceinline__ void run(float2* v) {
        float2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};
template <> struct Bfly<4> {
    static __device__ __forceinline__ void run(float2* v) {
        float2 a0 = cadd(v[0], v[2]), a1 = csub(v[0], v[2]);
        float2 a2 = cadd(v[1], v[3]), a3 = cmul_mi(csub(v[1], v[3]));
        v[0] = cadd(a0, a2);
        v[1] = cadd(a1, a3);
        v[2] = csub(a0, a2);
        v[3] = csub(a1, a3);
    }
};
template <> struct Bfly<8> {
    static __device__ __forceinline__ void run(float2* v) {
        float2 e[4] = {v[0], v[2], v[4], v[6]};
        float2 o[4] = {v[1], v[3], v[5], v[7]};
        Bfly<4>::run(e);
        Bfly<4>::run(o);
        const float c = 0.70710678118654752440f;
        float2 t1 = make_float2(c * (o[1].x + o[1].y), c * (o[1].y - o[1].x));    // o1 * (c, -c)
        float2 t2 = cmul_mi(o[2]);                                                // o2 * (-i)
        float2 t3 = make_float2(c * (o[3].y - o[3].x), -c * (o[3].x + o[3].y));   // o3 * (-c, -c)
        v[0] = cadd(e[0], o[0]); v[4] = csub(e[0], o[0]);
        v[1] = cadd(e[1], t1);   v[5] = csub(e[1], t1);
        v[2] = cadd(e[2], t2);   v[6] = csub(e[2], t2);
        v[3] = cadd(e[3], t3);   v[7] = csub(e[3], t3);
    }
};
template <> struct Bfly<16> {
    static __device__ __forceinline__ void run(float2* v) {
        float2 f[4][4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            f[r][0] = v[r]; f[r][1] = v[r + 4]; f[r][2] = v[r + 8]; f[r][3] = v[r + 12];
            Bfly<4>::run(f[r]);
        }
        // W16^m = (cos(pi m/8), -sin(pi m/8))
        const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f, c2 = 0.70710678118654752440f;
        const float2 W1 = make_float2(c1, -s1), W2 = make_float2(c2, -c2), W3 = make_float2(s1, -c1);
        const float2 W6 = make_float2(-c2, -c2), W9 = make_float2(-c1, s1);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            float2 t[4];
            t[0] = f[0][k];
            if (k == 0) { t[1] = f[1][0]; t[2] = f[2][0]; t[3] = f[3][0]; }
            if (k == 1) { t[1] = cmul(f[1][1], W1); t[2] = cmul(f[2][1], W2); t[3] = cmul(f[3][1], W3); }
            if (k == 2) { t[1] = cmul(f[1][2], W2); t[2] = cmul_mi(f[2][2]);  t[3] = cmul(f[3][2], W6); }
            if (k == 3) { t[1] = cmul(f[1][3], W3); t[2] = cmul(f[2][3], W6); t[3] = cmul(f[3][3], W9); }
            Bfly<4>::run(t);
            v[k] = t[0]; v[k + 4] = t[1]; v[k + 8] = t[2]; v[k + 12] = t[3];
        }
    }
};

// multiply v[k] by w^k, k = 1..R-1; powers built by a product tree of depth <= log2 R
template <int R>
__device__ __forceinline__ void twiddle_powers(float2* v, float2 w) {
    float2 p[R];
    p[1] = w;
#pragma unroll
    for (int k = 2; k < R; ++k) {
        int hi = 1;
        while (hi * 2 <= k) hi *= 2;
        p[k] = (hi == k) ? cmul(p[k / 2], p[k / 2]) : cmul(p[hi], p[k - hi]);
    }
#pragma unroll
    for (int k = 1; k < R; ++k) v[k] = cmul(v[k], p[k]);
}

// ------------------------------------------------------------------------------------------------------------
// per-length plan: radices, elements per thread, shared-memory padding (in complex elements) per exchange
//   PC1/PC2: pads of exchange 1/2 for the contiguous-line layout;  PS1/PS2: same for the strided layout with T lines
//   interleaved (element stride T);  TS: lines per CTA of the strided kernels;  LC: lines per CTA, contiguous kernels
// ------------------------------------------------------------------------------------------------------------
template <int K> struct Rad;
template <> struct Rad<32>   { static constexpr int R1 = 8,  R2 = 4,  R3 = 1, E = 8,  PC1 = 1, PC2 = 0, PS1 = 0, PS2 = 0, TS = 16, LC = 32, MBS = 1; };
template <> struct Rad<64>   { static constexpr int R1 = 8,  R2 = 8,  R3 = 1, E = 8,  PC1 = 1, PC2 = 0, PS1 = 0, PS2 = 0, TS = 16, LC = 32, MBS = 1; };
template <> struct Rad<128>  { static constexpr int R1 = 16, R2 = 8,  R3 = 1, E = 16, PC1 = 1, PC2 = 0, PS1 = 0, PS2 = 0, TS = 16, LC = 32, MBS = 1; };
template <> struct Rad<256>  { static constexpr int R1 = 16, R2 = 16, R3 = 1, E = 16, PC1 = 1, PC2 = 0, PS1 = 0, PS2 = 0, TS = 16, LC = 16, MBS = 4; };
template <> struct Rad<512>  { static constexpr int R1 = 8,  R2 = 8,  R3 = 8, E = 8,  PC1 = 8, PC2 = 1, PS1 = 0, PS2 = 1, TS = 8,  LC = 4, MBS = 3;  };
template <> struct Rad<1024> { static constexpr int R1 = 16, R2 = 8,  R3 = 8, E = 16, PC1 = 8, PC2 = 1, PS1 = 0, PS2 = 1, TS = 8,  LC = 4, MBS = 1;  };

template <int K> struct FftGeom {
    using C = Rad<K>;
    static constexpr int NS = (C::R3 > 1) ? 3 : 2;
    static constexpr int TPL = K / C::E;                                   // threads per line
    static constexpr int B1 = K / C::R1;                                   // exchange-1 nB range
    static constexpr int B2 = K / (C::R1 * C::R2);                         // exchange-2 nB range
    // contiguous layout: pitch in complex elements per line (kept = 8 mod 16 so that half-warps spanning two lines
    // fall into different bank halves)
    static constexpr int need_c1 = C::R1 * (B1 + C::PC1);
    static constexpr int need_c2 = (NS == 3) ? C::R1 * C::R2 * (B2 + C::PC2) : 0;
    static constexpr int need_c = need_c1 > need_c2 ? need_c1 : need_c2;
    static constexpr int PITCH_C = need_c + ((8 - need_c % 16) + 16) % 16;
    static constexpr int need_s1 = C::R1 * (B1 + C::PS1);
    static constexpr int need_s2 = (NS == 3) ? C::R1 * C::R2 * (B2 + C::PS2) : 0;
    static constexpr int SIZE_S = need_s1 > need_s2 ? need_s1 : need_s2;   // per line, strided layout
};

// Layout policies: physical shared-memory index of exchange element (kA, nB).
template <int K> struct LayContig {
    float2* base;   // start of this line's region
    __device__ __forceinline__ float2& ex1(int kA, int nB) const { return base[kA * (FftGeom<K>::B1 + Rad<K>::PC1) + nB]; }
    __device__ __forceinline__ float2& ex2(int kA, int nB) const { return base[kA * (FftGeom<K>::B2 + Rad<K>::PC2) + nB]; }
};
template <int K, int T> struct LayStrided {
    float2* base;   // smem base + t
    __device__ __forceinline__ float2& ex1(int kA, int nB) const { return base[(kA * (FftGeom<K>::B1 + Rad<K>::PS1) + nB) * T]; }
    __device__ __forceinline__ float2& ex2(int kA, int nB) const { return base[(kA * (FftGeom<K>::B2 + Rad<K>::PS2) + nB) * T]; }
};

// ------------------------------------------------------------------------------------------------------------
// One line.  q0 = thread index within the line (0..TPL-1).  ld(i) returns input element i, st(i, v) stores output
// element i.  PIN: inputs with index in [K/4, 3K/4) are known zero (never loaded).  POUT: outputs in [K/4, 3K/4) are
// not needed (never computed / stored).  tw = table of W_K^m = exp(-2 pi i m / K), m = 0..K-1 (float64-built).
// All threads of the CTA must call this together (it contains __syncthreads()).
// ------------------------------------------------------------------------------------------------------------
template <int K, bool PIN, bool POUT, class Lay, class Ld, class St>
__device__ __forceinline__ void fft_line(int q0, bool active, const Lay& lay, const float2* __restrict__ tw,
                                         const Ld& ld, const St& st) {
    using C = Rad<K>;
    using G = FftGeom<K>;
    constexpr int E = C::E, TPL = G::TPL;
    float2 v[E];

    // ---- stage 1: radix R1, A = 1, B = K/R1; butterfly id q = nB
    {
        constexpr int R = C::R1, B = K / R, NBF = E / R;
#pragma unroll
        for (int m = 0; m < NBF; ++m) {
            const int q = q0 + TPL * m;
#pragma unroll
            for (int n = 0; n < R; ++n) {
                const bool zero = PIN && (n >= R / 4) && (n < 3 * R / 4);
                v[m * R + n] = (zero || !active) ? make_float2(0.f, 0.f) : ld(q + n * B);
            }
        }
#pragma unroll
        for (int m = 0; m < NBF; ++m) {
            const int q = q0 + TPL * m;
            Bfly<R>::run(&v[m * R]);
            twiddle_powers<R>(&v[m * R], __ldg(&tw[q]));       // W_K^{nB k}
#pragma unroll
            for (int k = 0; k < R; ++k) lay.ex1(k, q) = v[m * R + k];
        }
    }
    __syncthreads();
    // ---- stage 2: radix R2, A = R1, B = K/(R1 R2)
    {
        constexpr int R = C::R2, A = C::R1, B = K / (A * R), NBF = E / R;
        constexpr bool LAST = (G::NS == 2);
#pragma unroll
        for (int m = 0; m < NBF; ++m) {
            const int q = q0 + TPL * m;
            const int kA = LAST ? q : q / B, nB = LAST ? 0 : q % B;
#pragma unroll
            for (int n = 0; n < R; ++n) v[m * R + n] = lay.ex1(kA, n * B + nB);
        }
        if (!LAST) __syncthreads();       // exchange buffer is reused
#pragma unroll
        for (int m = 0; m < NBF; ++m) {
            const int q = q0 + TPL * m;
            const int kA = LAST ? q : q / B, nB = LAST ? 0 : q % B;
            Bfly<R>::run(&v[m * R]);
            if (LAST) {
#pragma unroll
                for (int k = 0; k < R; ++k) {
                    const bool skip = POUT && (k >= R / 4) && (k < 3 * R / 4);
                    if (!skip && active) st(kA + A * k, v[m * R + k]);
                }
            } else {
                twiddle_powers<R>(&v[m * R], __ldg(&tw[nB * A]));   // W_K^{A nB k}
#pragma unroll
                for (int k = 0; k < R; ++k) lay.ex2(kA + A * k, nB) = v[m * R + k];
            }
        }
    }
    if constexpr (G::NS == 3) {
        __syncthreads();
        // ---- stage 3: radix R3, A = R1 R2, B = 1; butterfly id q = kA
        constexpr int R = C::R3, A = C::R1 * C::R2, NBF = E / R;
#pragma unroll
        for (int m = 0; m < NBF; ++m) {
            const int q = q0 + TPL * m;
#pragma unroll
            for (int n = 0; n < R; ++n) v[m * R + n] = lay.ex2(q, n);
        }
#pragma unroll
        for (int m = 0; m < NBF; ++m) {
            const int q = q0 + TPL * m;
            Bfly<R>::run(&v[m * R]);
#pragma unroll
            for (int k = 0; k < R; ++k) {
                const bool skip = POUT && (k >= R / 4) && (k < 3 * R / 4);
                if (!skip && active) st(q + A * k, v[m * R + k]);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Kernel parameters
// ------------------------------------------------------------------------------------------------------------
// Contiguous-line passes (the last image / grid axis).  A "line" is one row of the last axis.  Lines are numbered
// l = (b * n_outer0 + o0) * n_outer1 + o1 where o0, o1 run over the NON-ZERO (forward) / KEPT (adjoint) rows of the
// outer axes in image order; their grid coordinate is (o - N/2) mod K (circular placement, reading R4).
struct RowPassParams {
    const float2* img_in;     // forward: image x [batch][N0][N1]([N2]);  adjoint: unused
    float2* img_out;          // adjoint: image out;                      forward: unused
    float2* grid;             // workspace grid [batch][K0][K1]([K2])
    const float2* coil;       // optional coil maps [ncoil][prod N] (batch index = coil index), or nullptr
    const float* s_outer0;    // scaling vector of outer axis 0 (length n_outer0)
    const float* s_outer1;    // scaling vector of outer axis 1 (length n_outer1) or nullptr when d == 2
    const float* s_line;      // scaling vector of the line axis (length N)
    const float2* tw;
    int n_outer0, n_outer1;   // N of the outer axes (n_outer1 = 1 when d == 2)
    int k_outer0, k_outer1;   // K of the outer axes
    int nlines;               // batch * n_outer0 * n_outer1
    int img_batch_stride_is_zero;   // 1: the same image is used for every batch item (multi-coil forward)
};

// forward first pass: x (scaled, circularly zero-padded) -> FFT along the last axis -> grid rows
template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::LC)
fft_rows_fwd_kernel(RowPassParams p) {
    pdl_enter();
    using G = FftGeom<K>;
    constexpr int N = K / 2, TPL = G::TPL, LC = Rad<K>::LC;
    extern __shared__ float2 smem[];
    const int lt = threadIdx.x / TPL, q0 = threadIdx.x % TPL;
    const int line = blockIdx.x * LC + lt;
    const bool active = line < p.nlines;
    const int l = active ? line : 0;
    const int o1 = l % p.n_outer1, o0 = (l / p.n_outer1) % p.n_outer0, b = l / (p.n_outer1 * p.n_outer0);
    const int64_t img_line = ((int64_t)(p.img_batch_stride_is_zero ? 0 : b) * p.n_outer0 + o0) * p.n_outer1 + o1;
    const int64_t coil_line = ((int64_t)b * p.n_outer0 + o0) * p.n_outer1 + o1;
    const int g0 = (o0 - p.n_outer0 / 2) & (p.k_outer0 - 1), g1 = (o1 - p.n_outer1 / 2) & (p.k_outer1 - 1);
    const float2* __restrict__ src = p.img_in + img_line * N;
    const float2* __restrict__ csrc = p.coil ? p.coil + coil_line * N : nullptr;
    float2* __restrict__ dst = p.grid + (((int64_t)b * p.k_outer0 + g0) * p.k_outer1 + g1) * K;
    const float so = __ldg(&p.s_outer0[o0]) * (p.s_outer1 ? __ldg(&p.s_outer1[o1]) : 1.0f);
    const float* __restrict__ sl = p.s_line;
    LayContig<K> lay{smem + lt * G::PITCH_C};
    auto ld = [&](int i) -> float2 {
        const int n = (i + N / 2) & (K - 1);          // grid index i holds image sample n (i = (n - N/2) mod K)
        float2 xv = __ldg(&src[n]);
        if (csrc) xv = cmul(xv, __ldg(&csrc[n]));
        return cscale(xv, so * __ldg(&sl[n]));
    };
    auto st = [&](int i, float2 v) { dst[i] = v; };
    fft_line<K, true, false>(q0, active, lay, p.tw, ld, st);
}

// adjoint last pass: grid rows -> inverse FFT along the last axis -> crop -> S^H -> image
template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::LC)
fft_rows_adj_kernel(RowPassParams p) {
    pdl_enter();
    using G = FftGeom<K>;
    constexpr int N = K / 2, TPL = G::TPL, LC = Rad<K>::LC;
    extern __shared__ float2 smem[];
    const int lt = threadIdx.x / TPL, q0 = threadIdx.x % TPL;
    const int line = blockIdx.x * LC + lt;
    const bool active = line < p.nlines;
    const int l = active ? line : 0;
    const int o1 = l % p.n_outer1, o0 = (l / p.n_outer1) % p.n_outer0, b = l / (p.n_outer1 * p.n_outer0);
    const int64_t img_line = ((int64_t)b * p.n_outer0 + o0) * p.n_outer1 + o1;
    const int g0 = (o0 - p.n_outer0 / 2) & (p.k_outer0 - 1), g1 = (o1 - p.n_outer1 / 2) & (p.k_outer1 - 1);
    const float2* __restrict__ src = p.grid + (((int64_t)b * p.k_outer0 + g0) * p.k_outer1 + g1) * K;
    float2* __restrict__ dst = p.img_out + img_line * N;
    const float2* __restrict__ csrc = p.coil ? p.coil + img_line * N : nullptr;
    const float so = __ldg(&p.s_outer0[o0]) * (p.s_outer1 ? __ldg(&p.s_outer1[o1]) : 1.0f);
    const float* __restrict__ sl = p.s_line;
    LayContig<K> lay{smem + lt * G::PITCH_C};
    auto ld = [&](int i) -> float2 { return cconj(src[i]); };
    auto st = [&](int i, float2 v) {
        const int n = (i + N / 2) & (K - 1);
        float2 r = cscale(cconj(v), so * __ldg(&sl[n]));
        if (csrc) r = cmul(r, cconj(__ldg(&csrc[n])));      // conj(c_i) . A^H y_i   (eq. 35)
        dst[n] = r;
    };
    fft_line<K, false, true>(q0, active, lay, p.tw, ld, st);
}

// Strided passes (any axis but the last), in place on the grid.  A CTA transforms T lines that are adjacent in
// memory.  Group g -> (b, o, i0): element e of line t lives at  b*batch_stride + map(o)*outer_stride + e*line_stride
// + i0 + t,  map(o) = (o - n_outer/2) mod k_outer when the outer axis is pruned, else o.
struct ColPassParams {
    float2* grid;
    const float2* tw;
    int64_t batch_stride, outer_stride, line_stride;
    int n_outer, k_outer;      // number of outer slabs visited and K of that axis (k_outer = 0: identity map)
    int inner;                 // contiguous extent (multiple of T)
    int ngroups;               // batch * n_outer * inner / T
    const float2* mult;        // ADJ only, optional: every loaded element is first multiplied by mult[(offset within one
    int mult_shift;            //   batch item) >> mult_shift]  (Toeplitz spectrum; shift 5 on the interleaved grid)
};

// FULL: no pruning (every input is loaded, every output stored): used once per plan to transform the Toeplitz
// point-spread function, which fills the whole grid.
template <int K, bool ADJ, bool FULL = false, bool MULT = false>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::TS, Rad<K>::MBS)
fft_cols_kernel(ColPassParams p) {
    pdl_enter();
    using G = FftGeom<K>;
    constexpr int T = Rad<K>::TS;
    extern __shared__ float2 smem[];
    const int t = threadIdx.x % T, q0 = threadIdx.x / T;
    const int g = blockIdx.x;
    const int per_slab = p.inner / T;
    const int i0 = (g % per_slab) * T;
    const int o = (g / per_slab) % p.n_outer, b = g / (per_slab * p.n_outer);
    const int om = p.k_outer ? ((o - p.n_outer / 2) & (p.k_outer - 1)) : o;
    const int64_t off = (int64_t)om * p.outer_stride + i0 + t;
    float2* __restrict__ base = p.grid + (int64_t)b * p.batch_stride + off;
    const int64_t ls = p.line_stride;
    LayStrided<K, T> lay{smem + t};
    if (FULL) {
        auto ld = [&](int i) -> float2 { return base[i * ls]; };
        auto st = [&](int i, float2 v) { base[i * ls] = v; };
        fft_line<K, false, false>(q0, true, lay, p.tw, ld, st);
    } else if (!ADJ) {
        auto ld = [&](int i) -> float2 { return base[i * ls]; };
        auto st = [&](int i, float2 v) { base[i * ls] = v; };
        fft_line<K, true, false>(q0, true, lay, p.tw, ld, st);
    } else {
        const float2* __restrict__ mult = p.mult;
        const int ms = p.mult_shift;
        auto ld = [&](int i) -> float2 {
            float2 v = base[i * ls];
            if (MULT) v = cmul(v, __ldg(&mult[(off + i * ls) >> ms]));
            return cconj(v);
        };
        auto st = [&](int i, float2 v) { base[i * ls] = cconj(v); };
        fft_line<K, false, true>(q0, true, lay, p.tw, ld, st);
    }
}

// Unpruned in-place forward FFT along the last (contiguous) axis of a planar array: nlines lines of K elements.
template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::LC)
fft_rows_full_kernel(float2* __restrict__ data, const float2* __restrict__ tw, int nlines) {
    using G = FftGeom<K>;
    constexpr int TPL = G::TPL, LC = Rad<K>::LC;
    extern __shared__ float2 smem[];
    const int lt = threadIdx.x / TPL, q0 = threadIdx.x % TPL;
    const int line = blockIdx.x * LC + lt;
    const bool active = line < nlines;
    float2* __restrict__ row = data + (int64_t)(active ? line : 0) * K;
    LayContig<K> lay{smem + lt * G::PITCH_C};
    auto ld = [&](int i) -> float2 { return row[i]; };
    auto st = [&](int i, float2 v) { row[i] = v; };
    fft_line<K, false, false>(q0, active, lay, tw, ld, st);
}

// ------------------------------------------------------------------------------------------------------------
// Oversampling ratios other than 2 (SURVEY 8(f)-4 "other sigma"): any even N < K.  The pruned passes above hard-wire
// K = 2 N (the zero half is a radix digit), so these plans run the UNPRUNED FFT (fft_cols_kernel<K, false, true> for the
// strided axes) with S + zero-pad and crop + S^H fused into the contiguous-axis pass (fft_rows_pad_kernel /
// fft_rows_crop_kernel below).  F^H needs no conjugation pass: sum_k g_k e^{+i gamma k p} = FFT(g)[(-p) mod K].
// ------------------------------------------------------------------------------------------------------------
struct PadGeom {
    int d;
    int N[3], K[3];
    const float* s[3];       // scaling vectors per axis (length N[a])
};

// ------------------------------------------------------------------------------------------------------------
// sigma != 2 with S + zero-pad and crop + S^H FUSED into the contiguous-axis pass (round 2): the padded grid is never
// written by a separate pass and the cropped image never read back from one.
//   forward: fft_rows_pad_kernel runs over ALL grid lines; the loader maps the line's grid coordinates to image samples
//            (zero outside the image: such lines come out as zeros) and scales; unpruned FFT along the line.
//   adjoint: the strided passes run first (unpruned, in place); fft_rows_crop_kernel then transforms only the lines the crop
//            keeps and stores only the N kept outputs of each, at the reversed index (F^H through the forward FFT), scaled.
// ------------------------------------------------------------------------------------------------------------
struct SigmaRowParams {
    PadGeom g;
    const float2* img_in;     // forward: x [batch][prod N]
    float2* img_out;          // adjoint: x out
    float2* grid;             // [batch][prod K]
    const float2* coil;       // optional [batch][prod N]
    const float2* tw;         // twiddles of the line axis
    int64_t cells, nimg;
    int same_image;           // forward: every batch item reads image 0
    int nlines;               // forward: batch * prod(K outer);  adjoint: batch * prod(N outer)
};

// image index of grid coordinate k on an axis of size (N, K), or -1 in the zero-padded part
__device__ __forceinline__ int pad_map(int k, int N, int K) {
    const int h = N / 2;
    return (k < h) ? k + h : ((k >= K - h) ? k - K + h : -1);
}

template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::LC)
fft_rows_pad_kernel(SigmaRowParams p) {
    pdl_enter();
    using G = FftGeom<K>;
    constexpr int TPL = G::TPL, LC = Rad<K>::LC;
    extern __shared__ float2 smem[];
    const int lt = threadIdx.x / TPL, q0 = threadIdx.x % TPL;
    const int line = blockIdx.x * LC + lt;
    const bool active = line < p.nlines;
    const int d = p.g.d, NL = p.g.N[d - 1];
    // line -> (b, outer grid coordinates) -> outer image coordinates (or a zero line)
    int r = active ? line : 0;
    int64_t img_off = 0, mul = NL;
    float so = 1.0f;
    bool zero_line = false;
    for (int a = d - 2; a >= 0; --a) {
        const int k = r % p.g.K[a];
        r /= p.g.K[a];
        const int n = pad_map(k, p.g.N[a], p.g.K[a]);
        if (n < 0) zero_line = true;
        else { so *= __ldg(&p.g.s[a][n]); img_off += (int64_t)n * mul; }
        mul *= p.g.N[a];
    }
    const int b = r;
    const float2* __restrict__ src = p.img_in + (p.same_image ? 0 : (int64_t)b * p.nimg) + img_off;
    const float2* __restrict__ csrc = p.coil ? p.coil + (int64_t)b * p.nimg + img_off : nullptr;
    float2* __restrict__ dst = p.grid + (int64_t)(active ? line : 0) * K;
    const float* __restrict__ sl = p.g.s[d - 1];
    LayContig<K> lay{smem + lt * G::PITCH_C};
    auto ld = [&](int i) -> float2 {
        const int n = pad_map(i, NL, K);
        if (zero_line || n < 0) return make_float2(0.f, 0.f);
        float2 xv = __ldg(&src[n]);
        if (csrc) xv = cmul(xv, __ldg(&csrc[n]));
        return cscale(xv, so * __ldg(&sl[n]));
    };
    auto st = [&](int i, float2 v) { dst[i] = v; };
    fft_line<K, false, false>(q0, active, lay, p.tw, ld, st);
}

template <int K>
__global__ void __launch_bounds__(FftGeom<K>::TPL * Rad<K>::LC)
fft_rows_crop_kernel(SigmaRowParams p) {
    pdl_enter();
    using G = FftGeom<K>;
    constexpr int TPL = G::TPL, LC = Rad<K>::LC;
    extern __shared__ float2 smem[];
    const int lt = threadIdx.x / TPL, q0 = threadIdx.x % TPL;
    const int line = blockIdx.x * LC + lt;
    const bool active = line < p.nlines;
    const int d = p.g.d, NL = p.g.N[d - 1];
    // line -> (b, outer image coordinates) -> outer grid coordinates at the reversed index (-(n - N/2)) mod K
    int r = active ? line : 0;
    int64_t img_off = 0, imul = NL, cell_off = 0, cmul_ = K;
    float so = 1.0f;
    for (int a = d - 2; a >= 0; --a) {
        const int n = r % p.g.N[a];
        r /= p.g.N[a];
        const int k = (p.g.N[a] / 2 - n) & (p.g.K[a] - 1);
        so *= __ldg(&p.g.s[a][n]);
        img_off += (int64_t)n * imul;
        cell_off += (int64_t)k * cmul_;
        imul *= p.g.N[a];
        cmul_ *= p.g.K[a];
    }
    const int b = r;
    const float2* __restrict__ src = p.grid + (int64_t)b * p.cells + cell_off;
    float2* __restrict__ dst = p.img_out + (int64_t)b * p.nimg + img_off;
    const float2* __restrict__ csrc = p.coil ? p.coil + (int64_t)b * p.nimg + img_off : nullptr;
    const float* __restrict__ sl = p.g.s[d - 1];
    LayContig<K> lay{smem + lt * G::PITCH_C};
    auto ld = [&](int i) -> float2 { return src[i]; };
    auto st = [&](int i, float2 v) {
        const int n = (NL / 2 - i) & (K - 1);        // output i of the forward FFT is image sample n = (N/2 - i) mod K
        if (n < NL) {
            float2 o = cscale(v, so * __ldg(&sl[n]));
            if (csrc) o = cmul(o, cconj(__ldg(&csrc[n])));
            dst[n] = o;
        }
    };
    fft_line<K, false, false>(q0, active, lay, p.tw, ld, st);
}

}  // namespace nufft
