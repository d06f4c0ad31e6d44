"""Float64 CPU oracle of the NUFFT with the MIN-MAX interpolator.   TEST INFRASTRUCTURE.

PAPER.md:52, 74: "the default kernel is the min-max kernel [5]"; the paper prints no formula.  SURVEY.md 8(c) row 1 /
8(f)-4 fix the variant: min-max coefficients WITH THE KAISER-BESSEL SCALING FACTORS of oracle/nufft_oracle.py, so S, F,
F^H, S^H are unchanged and only the J interpolation weights per sample and axis differ.  Reading R25:

  Criterion of [5]: for a sample at u = om K / 2 pi with stencil k0 .. k0+J-1 (k0 = ceil(u - J/2), reading R6), choose the
  weights w that minimise the worst-case error over unit-norm images,
        max_{|x| = 1} | sum_p x_p ( e^{-i om p} - s_p sum_j w_j e^{-i gamma (k0 + j) p} ) |  =  || 1 - diag(s) C w ||_2 ,
  C[p, j] = e^{ i gamma t_j p },  t_j = u - k0 - j,  gamma = 2 pi / K  (Cauchy-Schwarz: the worst case IS the 2-norm),
  i.e. a linear least-squares problem per sample:  T w = r,
        T[l, j] = sum_p c_p s_p^2 cos(gamma (l - j) p),      r[l] = sum_p c_p s_p cos(gamma t_l p).
  Pixel set and REAL weights: the image occupies positions p = n - N/2 in [-N/2, N/2) (reading R4), which is not symmetric
  about 0, so the unrestricted least-squares solution is slightly complex.  The hot path carries real, separable weights
  (readings R3/R4 make the Kaiser-Bessel weights real), so R25 takes the minimiser over REAL weight vectors: stacking
  real and imaginary rows gives exactly the cosine sums above over the image's own N pixels.  Because the summands are
  even in p this equals the sum over the symmetric set p = -N/2 .. N/2 with weight c = 1/2 on both end points, which is
  how it is written below.  (The unrestricted complex optimum has a worst-case error up to ~1.4x smaller at N = 16; [5]'s
  own centring (N-1)/2 is the other way to real weights and would move the image by half a pixel, contradicting R4.)

Follows the algorithm step by step; library primitives: numpy.linalg.solve (the J x J system), numpy.fft through
nufft_oracle.scale_pad_fft / ifft_crop_scale, numpy.bincount through nufft_oracle.grid_adjoint.

Parity pins (tests/test_oracle_minmax.py, `-m "not gpu"`): the normal equations checked with explicitly assembled complex
matrices (best real weight vector of the image's own pixel set; residual orthogonal to the columns); the error vector
shown to be the error of the transform; the worst-case error not larger than the Kaiser-Bessel weights' on the same stencil; brute-force NDFT (<= 1e-4, north star); adjoint identity;
mirror symmetry w_j(t) = w_{J-1-j}(-t).  No function here is "parity unpinned".
"""
import numpy as np

from . import nufft_oracle as orc

__all__ = ["minmax_T", "minmax_weights", "stencil", "interp", "grid_adjoint", "forward", "adjoint", "selfadjoint"]


def _pixels(N):
    """Symmetric pixel set p = -N/2 .. N/2 and its weights c (1/2 on the two end points)."""
    p = np.arange(-(N // 2), N // 2 + 1, dtype=np.float64)
    c = np.ones(p.size)
    c[0] = c[-1] = 0.5
    return p, c


def _s_of_p(p, N, K, J):
    """Kaiser-Bessel scaling factor at pixel position p (even in p): 1 / Phi(p / K)  (reading R3)."""
    beta = orc.kb_beta(J, K / N)
    return 1.0 / orc.kb_Phi(p / K, J, beta)


def minmax_T(N, K, J):
    """T[l, j] = sum_p c_p s_p^2 cos(gamma (l - j) p): J x J, symmetric Toeplitz, the same for every sample of an axis."""
    p, c = _pixels(N)
    s = _s_of_p(p, N, K, J)
    gam = 2.0 * np.pi / K
    lj = np.arange(J)[:, None] - np.arange(J)[None, :]
    return np.einsum("p,ljp->lj", c * s * s, np.cos(gam * lj[:, :, None] * p[None, None, :]))


def minmax_weights(t, N, K, J, chunk=2048):
    """Weights of the samples whose stencil offsets are t[M][J] (t_j = u - k0 - j, grid cells): solve T w = r(t)."""
    t = np.asarray(t, dtype=np.float64)
    p, c = _pixels(N)
    cs = c * _s_of_p(p, N, K, J)
    gam = 2.0 * np.pi / K
    T = minmax_T(N, K, J)
    w = np.empty_like(t)
    for a in range(0, t.shape[0], chunk):
        tt = t[a:a + chunk]
        r = np.cos(gam * tt[:, :, None] * p[None, None, :]) @ cs            # [m][J]
        w[a:a + chunk] = np.linalg.solve(T, r.T).T
    return w


def stencil(om_a, N, K, J):
    """Per-axis stencil: the grid indices of nufft_oracle.stencil (same k0, reading R6/R7), min-max weights."""
    om_a = np.asarray(om_a, dtype=np.float64)
    u = om_a * (K / (2.0 * np.pi))
    k0 = np.ceil(u - J / 2.0)
    j = np.arange(J, dtype=np.float64)
    idx = np.mod(k0[:, None] + j[None, :], K).astype(np.int64)
    t = u[:, None] - k0[:, None] - j[None, :]
    return idx, minmax_weights(t, N, K, J)


def _stencils(om, Nd, Kd, Jd):
    om = np.asarray(om, dtype=np.float64)
    return [stencil(om[:, a], Nd[a], Kd[a], Jd[a]) for a in range(len(Nd))]


def interp(G, om, Nd, Kd, Jd):
    """V with the min-max weights."""
    return orc.interp(G, om, Nd, Kd, Jd, st=_stencils(om, Nd, Kd, Jd))


def grid_adjoint(y, om, Nd, Kd, Jd):
    """V^H with the min-max weights."""
    return orc.grid_adjoint(y, om, Nd, Kd, Jd, st=_stencils(om, Nd, Kd, Jd))


def forward(x, om, Nd, Kd, Jd):
    """y = V_minmax F S x  (eq. 1)."""
    return interp(orc.scale_pad_fft(x, Nd, Kd, Jd), om, Nd, Kd, Jd)


def adjoint(y, om, Nd, Kd, Jd):
    """x = S^H F^H V_minmax^H y  (eq. 2)."""
    return orc.ifft_crop_scale(grid_adjoint(y, om, Nd, Kd, Jd), Nd, Kd, Jd)


def selfadjoint(x, om, Nd, Kd, Jd):
    """A^H A x, back to back (eq. 5; reading R8)."""
    return adjoint(forward(x, om, Nd, Kd, Jd), om, Nd, Kd, Jd)
