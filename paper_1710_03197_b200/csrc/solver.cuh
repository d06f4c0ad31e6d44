// solver.cuh -- elementwise / reduction glue of the solvers built on A^H A (step a9 of SURVEY.md 8(a)):
// conjugate gradient (reading R12) and split-Bregman L1TV-OLS (eqs. 12-22,
// readings R13-R18).  Images are complex64; every inner product and every CG scalar is float64 and stays on the
// device (only the plan is offloaded "before iterative algorithms begin"; nothing returns per iteration).
#pragma once
#include "common.cuh"

namespace nufft {

// device-resident CG scalars
struct CgScalars {
    double rs;        // <r, r> of the current residual
    double pAp;       // accumulator: Re <p, A p>
    double rs_new;    // accumulator: <r, r> after the update
    double maxabs;    // scratch for max |.| reductions (bit pattern of a non-negative double, ordered as int64)
    int hist_pos;     // next slot of the residual-norm history (kept on the device so that one iteration is one replayable graph)
};

__device__ __forceinline__ double block_reduce_sum(double v) {
    __shared__ double red[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? red[threadIdx.x] : 0.0;
    if (wid == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    }
    return v;   // valid in thread 0
}

// *out += Re <a, b> = sum Re(conj(a) b)
__global__ void __launch_bounds__(256)
dot_real_kernel(const float2* __restrict__ a, const float2* __restrict__ b, int64_t n, double* out) {
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float2 u = a[i], v = b[i];
        acc += (double)u.x * (double)v.x + (double)u.y * (double)v.y;
    }
    acc = block_reduce_sum(acc);
    if (threadIdx.x == 0) atomicAdd(out, acc);
}

// r = rhs - Ax;  p = r;  *rs += <r, r>
__global__ void __launch_bounds__(256)
cg_init_kernel(const float2* __restrict__ rhs, const float2* __restrict__ Ax, float2* __restrict__ r,
               float2* __restrict__ p, int64_t n, CgScalars* s) {
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        float2 v = rhs[i];
        if (Ax) v = csub(v, Ax[i]);
        r[i] = v;
        p[i] = v;
        acc += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
    }
    acc = block_reduce_sum(acc);
    if (threadIdx.x == 0) atomicAdd(&s->rs, acc);
}

// alpha = rs / pAp;  x += alpha p;  r -= alpha Ap;  *rs_new += <r, r>
__global__ void __launch_bounds__(256)
cg_update_xr_kernel(float2* __restrict__ x, float2* __restrict__ r, const float2* __restrict__ p,
                    const float2* __restrict__ Ap, int64_t n, CgScalars* s) {
    const double rs = s->rs, pAp = s->pAp;
    const float alpha = (rs == 0.0) ? 0.0f : (float)(rs / pAp);
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float2 pv = p[i], av = Ap[i];
        float2 xv = x[i], rv = r[i];
        xv.x = fmaf(alpha, pv.x, xv.x); xv.y = fmaf(alpha, pv.y, xv.y);
        rv.x = fmaf(-alpha, av.x, rv.x); rv.y = fmaf(-alpha, av.y, rv.y);
        x[i] = xv; r[i] = rv;
        acc += (double)rv.x * (double)rv.x + (double)rv.y * (double)rv.y;
    }
    acc = block_reduce_sum(acc);
    if (threadIdx.x == 0) atomicAdd(&s->rs_new, acc);
}

// beta = rs_new / rs;  p = r + beta p
__global__ void __launch_bounds__(256)
cg_update_p_kernel(float2* __restrict__ p, const float2* __restrict__ r, int64_t n, const CgScalars* s) {
    const double rs = s->rs, rsn = s->rs_new;
    const float beta = (rs == 0.0) ? 0.0f : (float)(rsn / rs);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float2 rv = r[i];
        float2 pv = p[i];
        pv.x = fmaf(beta, pv.x, rv.x); pv.y = fmaf(beta, pv.y, rv.y);
        p[i] = pv;
    }
}

// rs <- rs_new, accumulators cleared, residual norm logged
__global__ void cg_shift_kernel(CgScalars* s, double* hist, int first) {
    if (!first) s->rs = s->rs_new;
    s->rs_new = 0.0;
    s->pAp = 0.0;
    if (hist) hist[s->hist_pos++] = sqrt(s->rs);
}

__global__ void scalars_clear_kernel(CgScalars* s) { s->rs = 0.0; s->pAp = 0.0; s->rs_new = 0.0; s->maxabs = 0.0; s->hist_pos = 0; }

// max |a_i|  (non-negative doubles order like their bit patterns)
__global__ void __launch_bounds__(256)
maxabs_kernel(const float2* __restrict__ a, int64_t n, CgScalars* s) {
    float m = 0.f;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float2 v = a[i];
        m = fmaxf(m, v.x * v.x + v.y * v.y);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0)
        atomicMax((long long*)&s->maxabs, __double_as_longlong(sqrt((double)m)));
}

// out = a * s
__global__ void __launch_bounds__(256)
scale_kernel(float2* __restrict__ out, const float2* __restrict__ a, float sc, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        out[i] = cscale(a[i], sc);
}

// out = sum_i img[i]   (coil sum of eq. 35; the conj(c_i) factor was applied by the last adjoint FFT pass)
__global__ void __launch_bounds__(256)
coil_sum_kernel(float2* __restrict__ out, const float2* __restrict__ img, int ncoil, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        float2 acc = make_float2(0.f, 0.f);
        for (int c = 0; c < ncoil; ++c) acc = cadd(acc, img[(int64_t)c * n + i]);
        out[i] = acc;
    }
}

// ---- total-variation pieces, 2-D image [N0][N1], periodic forward difference (eq. 12, R15) ----
//   grad_a x = x(n + e_a) - x(n);   grad_a^T v = v(n - e_a) - v(n)

// out = mu * out + lam * sum_a grad_a^T grad_a z       (eq. 15: K z, with `out` holding A^H A z on entry)
__global__ void __launch_bounds__(256)
tv_normal_kernel(float2* __restrict__ out, const float2* __restrict__ z, float mu, float lam, int N0, int N1) {
    const int64_t n = (int64_t)N0 * N1;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int n0 = (int)(i / N1), n1 = (int)(i % N1);
        const float2 c = z[i];
        const float2 up = z[(int64_t)((n0 + 1) % N0) * N1 + n1], dn = z[(int64_t)((n0 + N0 - 1) % N0) * N1 + n1];
        const float2 rt = z[(int64_t)n0 * N1 + (n1 + 1) % N1], lf = z[(int64_t)n0 * N1 + (n1 + N1 - 1) % N1];
        // grad^T grad z = (z - z(-1)) - (z(+1) - z) per axis
        const float lx = (c.x - dn.x) - (up.x - c.x) + (c.x - lf.x) - (rt.x - c.x);
        const float ly = (c.y - dn.y) - (up.y - c.y) + (c.y - lf.y) - (rt.y - c.y);
        float2 o = out[i];
        o.x = fmaf(mu, o.x, lam * lx);
        o.y = fmaf(mu, o.y, lam * ly);
        out[i] = o;
    }
}

// rhs = mu * ahy + lam * sum_a grad_a^T (d_a - b_a)       (eq. 16)
__global__ void __launch_bounds__(256)
tv_rhs_kernel(float2* __restrict__ rhs, const float2* __restrict__ ahy, const float2* __restrict__ d0,
              const float2* __restrict__ b0, const float2* __restrict__ d1, const float2* __restrict__ b1,
              float mu, float lam, int N0, int N1) {
    const int64_t n = (int64_t)N0 * N1;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int n0 = (int)(i / N1), n1 = (int)(i % N1);
        const int64_t im0 = (int64_t)((n0 + N0 - 1) % N0) * N1 + n1, im1 = (int64_t)n0 * N1 + (n1 + N1 - 1) % N1;
        const float2 v0 = csub(d0[i], b0[i]), v0m = csub(d0[im0], b0[im0]);
        const float2 v1 = csub(d1[i], b1[i]), v1m = csub(d1[im1], b1[im1]);
        const float2 a = ahy[i];
        const float tx = (v0m.x - v0.x) + (v1m.x - v1.x), ty = (v0m.y - v0.y) + (v1m.y - v1.y);
        rhs[i] = make_float2(fmaf(lam, tx, mu * a.x), fmaf(lam, ty, mu * a.y));
    }
}

// d_a = shrink(grad_a x + b_a, thr);  b_a += grad_a x - d_a       (eqs. 18-21, readings R13, R14)
// shrink(z, t) = z max(|z| - t, 0) / |z|, 0 at z = 0.  thr < 0 encodes +infinity (lam = 0): d = 0.
__global__ void __launch_bounds__(256)
tv_shrink_kernel(const float2* __restrict__ x, float2* __restrict__ d0, float2* __restrict__ b0,
                 float2* __restrict__ d1, float2* __restrict__ b1, float thr, int N0, int N1) {
    const int64_t n = (int64_t)N0 * N1;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int n0 = (int)(i / N1), n1 = (int)(i % N1);
        const float2 c = x[i];
        const float2 g0 = csub(x[(int64_t)((n0 + 1) % N0) * N1 + n1], c);
        const float2 g1 = csub(x[(int64_t)n0 * N1 + (n1 + 1) % N1], c);
        {
            const float2 b = b0[i], t = cadd(g0, b);
            const float mag = sqrtf(t.x * t.x + t.y * t.y);
            const float f = (thr < 0.f || mag <= 0.f) ? 0.f : fmaxf(mag - thr, 0.f) / mag;
            const float2 dn = cscale(t, f);
            d0[i] = dn;
            b0[i] = cadd(b, csub(g0, dn));
        }
        {
            const float2 b = b1[i], t = cadd(g1, b);
            const float mag = sqrtf(t.x * t.x + t.y * t.y);
            const float f = (thr < 0.f || mag <= 0.f) ? 0.f : fmaxf(mag - thr, 0.f) / mag;
            const float2 dn = cscale(t, f);
            d1[i] = dn;
            b1[i] = cadd(b, csub(g1, dn));
        }
    }
}

// ahy_k += ahy_s - ahax       (eq. 22)
__global__ void __launch_bounds__(256)
tv_outer_kernel(float2* __restrict__ ahy_k, const float2* __restrict__ ahy_s, const float2* __restrict__ ahax, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        ahy_k[i] = cadd(ahy_k[i], csub(ahy_s[i], ahax[i]));
}

// ---- L1TV-LAD data-term split, eqs. (25), (29), (32) PAPER.md:224-243 (reading R23) ----
// out = ahy_k + d_f - b_f      (the bracket of eq. 25)
__global__ void __launch_bounds__(256)
lad_prep_kernel(float2* __restrict__ out, const float2* __restrict__ ahy_k, const float2* __restrict__ df,
                const float2* __restrict__ bf, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        out[i] = cadd(ahy_k[i], csub(df[i], bf[i]));
}
// r = A^H A x - A^H y;  d_f = shrink(r + b_f, thr);  b_f += r - d_f.   thr < 0 encodes +infinity (mu = 0): d_f = 0.
__global__ void __launch_bounds__(256)
lad_data_kernel(const float2* __restrict__ ahax, const float2* __restrict__ ahy_s, float2* __restrict__ df,
                float2* __restrict__ bf, float thr, int64_t n) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float2 r = csub(ahax[i], ahy_s[i]);
        const float2 b = bf[i], t = cadd(r, b);
        const float mag = sqrtf(t.x * t.x + t.y * t.y);
        const float f = (thr < 0.f || mag <= 0.f) ? 0.f : fmaxf(mag - thr, 0.f) / mag;
        const float2 dn = cscale(t, f);
        df[i] = dn;
        bf[i] = cadd(b, csub(r, dn));
    }
}

// ---- density compensation, eqs. (6)-(7) PAPER.md:118-122 (reading R21) ----
// w = 1 (complex64 with zero imaginary part)
__global__ void __launch_bounds__(256) dcf_init_kernel(float2* __restrict__ w, int64_t M) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < M; i += (int64_t)gridDim.x * blockDim.x)
        w[i] = make_float2(1.f, 0.f);
}
// w <- w / |t|,  t = A A^H w
__global__ void __launch_bounds__(256) dcf_update_kernel(float2* __restrict__ w, const float2* __restrict__ t, int64_t M) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < M; i += (int64_t)gridDim.x * blockDim.x) {
        const float2 tv = t[i];
        const float mag = sqrtf(tv.x * tv.x + tv.y * tv.y);
        // |A A^H w| = 0 (a sample no image pixel reaches: degenerate input): the weight becomes 0 instead of inf
        w[i] = make_float2(mag > 0.f ? w[i].x / mag : 0.f, 0.f);
    }
}
// out[b][m] = y[b][m] * w[m].re
__global__ void __launch_bounds__(256)
weight_mul_kernel(float2* __restrict__ out, const float2* __restrict__ y, const float2* __restrict__ w, int64_t M, int batch) {
    const int64_t n = M * batch;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        out[i] = cscale(y[i], __ldg(&w[i % M].x));
}

// grid[b][i] *= spec[i]   (1-D Toeplitz: there is no adjoint column pass to carry the spectrum multiply)
__global__ void __launch_bounds__(256)
spectrum_mul_kernel(float2* __restrict__ grid, const float2* __restrict__ spec, int64_t cells, int batch) {
    const int64_t n = cells * batch;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        grid[i] = cmul(grid[i], __ldg(&spec[i % cells]));
}

// ---- Toeplitz point-spread function (reading R22) ----
// T2 is the adjoint NUFFT of the weights onto the 2N image (pixel n <-> displacement d = n - N).  Zero the d = -N
// hyperplanes (pixel 0 of every axis), which a linear convolution of two length-N supports never uses.
__global__ void __launch_bounds__(256) psf_zero_planes_kernel(float2* __restrict__ T, int K0, int K1, int K2) {
    const int64_t n = (int64_t)K0 * K1 * K2;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int c2 = (int)(i % K2), c1 = (int)((i / K2) % K1), c0 = (int)(i / ((int64_t)K1 * K2));
        if (c0 == 0 || (K1 > 1 && c1 == 0) || (K2 > 1 && c2 == 0)) T[i] = make_float2(0.f, 0.f);
    }
}
// T[h N + n] = blk[n] per axis: one N^d block of the point-spread function into the (2N)^d array (R22)
__global__ void __launch_bounds__(256)
psf_place_block_kernel(float2* __restrict__ T, const float2* __restrict__ blk, int N0, int N1, int N2, int h0, int h1, int h2) {
    const int64_t n = (int64_t)N0 * N1 * N2;
    const int64_t K1 = 2 * (int64_t)N1, K2 = (N2 > 1) ? 2 * (int64_t)N2 : 1;
    const int64_t K1e = (N1 > 1) ? K1 : 1;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int n2 = (int)(i % N2), n1 = (int)((i / N2) % N1), n0 = (int)(i / ((int64_t)N1 * N2));
        const int64_t o = ((int64_t)(h0 * N0 + n0) * K1e + (h1 * N1 + n1)) * K2 + (h2 * N2 + n2);
        T[o] = blk[i];
    }
}

// T^[k] = sum_d T[d] e^{-2 pi i k d / K} = (-1)^{sum k_a} FFT(T2)[k]   (d = n - K/2 per axis), times `scale` = 1/prod(K):
// the path's F^H is the unnormalised conjugate transpose (R5), so F^H(T^ . F z) carries a factor prod(K).
__global__ void __launch_bounds__(256) psf_sign_kernel(float2* __restrict__ T, int K0, int K1, int K2, float scale) {
    const int64_t n = (int64_t)K0 * K1 * K2;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int c2 = (int)(i % K2), c1 = (int)((i / K2) % K1), c0 = (int)(i / ((int64_t)K1 * K2));
        const float sgn = ((c0 + c1 + c2) & 1) ? -scale : scale;
        T[i] = make_float2(sgn * T[i].x, sgn * T[i].y);
    }
}

}  // namespace nufft
