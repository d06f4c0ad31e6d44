"""Float64 CPU oracle of the three-stage NUFFT  A = V F S  and its adjoint.   TEST INFRASTRUCTURE.

Follows PAPER.md (arxiv 1710.03197) section 2.1 stage by stage, in the paper's order and notation:
    S   scaling                       PAPER.md:54-56   (section 2.1.1)
    F   zero-padding + oversampled FFT PAPER.md:58-68   (section 2.1.2)
    V   interpolation                 PAPER.md:72-74   (section 2.1.3)
    V^H gridding = conj. transpose of V PAPER.md:76
    A^H = S^H F^H V^H                 PAPER.md:78-84   (section 2.1.4, eq. 2)
    A^H A  (self-adjoint)             PAPER.md:86-98   (section 2.1.5, eq. 5)
    multi-coil                        PAPER.md:251-258 (eqs. 34-35)

The paper does not print the interpolator's formula ("min-max kernel [5], whereas other kernel functions
can be used").  Reading taken (readings R1-R7):
plain Kaiser-Bessel window of width J grid cells, real and separable, with the closed-form Fourier
transform as the scaling factor, forward sign e^{-i...}, image index n at position n - N/2, periodic grid,
unnormalised F^H (true conjugate transpose).

Everything is numpy float64 / complex128.  Library primitives used as steps: numpy.fft.fftn / ifftn (F, F^H),
numpy.i0 (modified Bessel I0), numpy.bincount (the scatter-add of V^H).

Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
    kb_phi, kb_Phi, scaling_factors   quadrature of the defining integral; I0 power series; closed-form values
    stencil / interp / grid_adjoint   dense M x prod(K) matrix on tiny sizes; partition of unity
    forward / adjoint                 brute-force non-uniform DFT (ndft_*), rel. L2 <= 1e-4; adjoint identity
                                      <Ax,y> = <x,A^H y> to 1e-10; unit-impulse closed form; Cartesian
                                      samples vs numpy.fft
    selfadjoint                       Hermitian / positive semi-definite; equals adjoint(forward(x))
    multi-coil                        explicit loop over coils
No function here is "parity unpinned".
"""
import numpy as np

__all__ = [
    "kb_beta", "kb_phi", "kb_Phi", "scaling_factors", "stencil", "interp", "grid_adjoint",
    "scale_pad_fft", "ifft_crop_scale", "forward", "adjoint", "selfadjoint",
    "forward_coils", "adjoint_coils", "selfadjoint_coils", "ndft_forward", "ndft_adjoint",
]


# ----------------------------------------------------------------------------------------------------------
# Interpolation kernel (reading R1/R2: Kaiser-Bessel, beta from the oversampling ratio)
# ----------------------------------------------------------------------------------------------------------
def kb_beta(J, sigma):
    """Shape parameter beta = pi * sqrt((J/sigma)^2 (sigma - 1/2)^2 - 0.8)  (reading R2).

    J = kernel width in grid cells, sigma = K/N oversampling ratio.  J=6, sigma=2 -> 13.8551003461...
    """
    J = float(J)
    sigma = float(sigma)
    return np.pi * np.sqrt((J / sigma) ** 2 * (sigma - 0.5) ** 2 - 0.8)


def kb_phi(t, J, beta):
    """phi(t) = I0(beta * sqrt(1 - (2t/J)^2)) / I0(beta) for |t| < J/2, else 0  (reading R1).

    t in grid cells.  phi(0) = 1.  The support is open: phi(+-J/2) = 0 (reading R6).
    """
    t = np.asarray(t, dtype=np.float64)
    a = 1.0 - (2.0 * t / float(J)) ** 2
    inside = (np.abs(t) < float(J) / 2.0) & (a > 0.0)
    val = np.i0(beta * np.sqrt(np.where(inside, a, 0.0))) / np.i0(beta)
    return np.where(inside, val, 0.0)


def kb_Phi(xi, J, beta):
    """Continuous Fourier transform of phi:  Phi(xi) = int phi(t) e^{-2 pi i xi t} dt
         = (J / I0(beta)) * sinh(z)/z,  z = sqrt(beta^2 - (pi J xi)^2)      (z^2 > 0)
         = (J / I0(beta)) * sin(z')/z', z' = sqrt((pi J xi)^2 - beta^2)     (z^2 < 0)
    xi in cycles per grid cell.
    """
    xi = np.asarray(xi, dtype=np.float64)
    z2 = beta ** 2 - (np.pi * float(J) * xi) ** 2
    zp = np.sqrt(np.abs(z2))
    small = zp < 1e-12
    zs = np.where(small, 1.0, zp)
    val = np.where(z2 >= 0.0, np.sinh(zs) / zs, np.sin(zs) / zs)
    val = np.where(small, 1.0, val)
    return float(J) / np.i0(beta) * val


def scaling_factors(N, K, J):
    """1-D scaling factors s[n] = 1 / Phi((n - N/2)/K), n = 0..N-1  (reading R3).

    Real and positive.  The d-dimensional S is the outer product of the per-axis vectors.
    """
    beta = kb_beta(J, K / N)
    n = np.arange(N, dtype=np.float64)
    return 1.0 / kb_Phi((n - N / 2.0) / K, J, beta)


# ----------------------------------------------------------------------------------------------------------
# V and V^H
# ----------------------------------------------------------------------------------------------------------
def stencil(om_a, N, K, J):
    """Per-axis stencil of every sample (reading R6).

    om_a[M] radians per image sample.  u = om * K / (2 pi);  k0 = ceil(u - J/2);  for j = 0..J-1:
    grid index (k0 + j) mod K (reading R7: periodic), weight phi(u - k0 - j).
    Returns idx[M][J] int64, w[M][J] float64.
    """
    om_a = np.asarray(om_a, dtype=np.float64)
    beta = kb_beta(J, K / N)
    u = om_a * (K / (2.0 * np.pi))
    k0 = np.ceil(u - J / 2.0)
    j = np.arange(J, dtype=np.float64)
    idx = np.mod(k0[:, None] + j[None, :], K).astype(np.int64)
    w = kb_phi(u[:, None] - k0[:, None] - j[None, :], J, beta)
    return idx, w


def _stencils(om, Nd, Kd, Jd):
    om = np.asarray(om, dtype=np.float64)
    d = len(Nd)
    assert om.ndim == 2 and om.shape[1] == d
    return [stencil(om[:, a], Nd[a], Kd[a], Jd[a]) for a in range(d)]


def _offsets(Jd):
    return np.ndindex(*[int(j) for j in Jd])


def interp(G, om, Nd, Kd, Jd, st=None):
    """V:  y[m] = sum_j  prod_a w_a[m, j_a] * G[(k0 + j) mod K].

    G has shape Kd (C order).  Returns y[M] complex128.  st: per-axis (idx, w) lists from another real, separable
    interpolator (oracle/minmax_oracle.py); default = the Kaiser-Bessel stencils of this module.
    """
    G = np.asarray(G, dtype=np.complex128)
    st = _stencils(om, Nd, Kd, Jd) if st is None else st
    M = st[0][0].shape[0]
    y = np.zeros(M, dtype=np.complex128)
    for j in _offsets(Jd):
        w = np.ones(M)
        index = []
        for a, ja in enumerate(j):
            w = w * st[a][1][:, ja]
            index.append(st[a][0][:, ja])
        y += w * G[tuple(index)]
    return y


def grid_adjoint(y, om, Nd, Kd, Jd, st=None):
    """V^H:  G[(k0 + j) mod K] += prod_a w_a[m, j_a] * y[m]   over all m, j.

    The weights are real, so the conjugate transpose of V has the same weights.  Returns G of shape Kd.  st as in interp.
    """
    y = np.asarray(y, dtype=np.complex128)
    st = _stencils(om, Nd, Kd, Jd) if st is None else st
    M = y.shape[0]
    size = int(np.prod(Kd))
    Gr = np.zeros(size)
    Gi = np.zeros(size)
    for j in _offsets(Jd):
        w = np.ones(M)
        index = []
        for a, ja in enumerate(j):
            w = w * st[a][1][:, ja]
            index.append(st[a][0][:, ja])
        flat = np.ravel_multi_index(tuple(index), tuple(int(k) for k in Kd))
        Gr += np.bincount(flat, weights=w * y.real, minlength=size)
        Gi += np.bincount(flat, weights=w * y.imag, minlength=size)
    return (Gr + 1j * Gi).reshape(tuple(int(k) for k in Kd))


# ----------------------------------------------------------------------------------------------------------
# S, zero-pad, F and their transposes
# ----------------------------------------------------------------------------------------------------------
def _pad_index(Nd, Kd):
    """Grid index of image sample n on each axis: (n - N/2) mod K (reading R4: circular placement)."""
    return np.ix_(*[np.mod(np.arange(N) - N // 2, K) for N, K in zip(Nd, Kd)])


def _S(Nd, Kd, Jd):
    s = np.ones(())
    for N, K, J in zip(Nd, Kd, Jd):
        s = np.multiply.outer(s, scaling_factors(N, K, J))
    return s


def scale_pad_fft(x, Nd, Kd, Jd):
    """F S x:  multiply by the scaling factors, copy into the zeroed Kd array, FFT."""
    x = np.asarray(x, dtype=np.complex128)
    g = np.zeros(tuple(int(k) for k in Kd), dtype=np.complex128)
    g[_pad_index(Nd, Kd)] = _S(Nd, Kd, Jd) * x
    return np.fft.fftn(g)


def ifft_crop_scale(G, Nd, Kd, Jd):
    """S^H F^H G:  unnormalised inverse FFT (reading R5), array copy (crop), rescale."""
    g = np.fft.ifftn(np.asarray(G, dtype=np.complex128)) * float(np.prod(Kd))
    return _S(Nd, Kd, Jd) * g[_pad_index(Nd, Kd)]


# ----------------------------------------------------------------------------------------------------------
# A, A^H, A^H A
# ----------------------------------------------------------------------------------------------------------
def forward(x, om, Nd, Kd, Jd):
    """y = A x = V F S x  (eq. 1).  x shape Nd -> y[M]."""
    return interp(scale_pad_fft(x, Nd, Kd, Jd), om, Nd, Kd, Jd)


def adjoint(y, om, Nd, Kd, Jd):
    """x = A^H y = S^H F^H V^H y  (eq. 2).  y[M] -> x shape Nd."""
    return ifft_crop_scale(grid_adjoint(y, om, Nd, Kd, Jd), Nd, Kd, Jd)


def selfadjoint(x, om, Nd, Kd, Jd):
    """A^H A x, applied back to back  (eq. 5; reading R8)."""
    return adjoint(forward(x, om, Nd, Kd, Jd), om, Nd, Kd, Jd)


def forward_coils(x, c, om, Nd, Kd, Jd):
    """A_multi x = [A (c_i . x)]_i   (eq. 35).  c[Nc, *Nd] -> y[Nc, M]."""
    return np.stack([forward(ci * x, om, Nd, Kd, Jd) for ci in c])


def adjoint_coils(y, c, om, Nd, Kd, Jd):
    """A_multi^H y = sum_i conj(c_i) . A^H y_i   (eqs. 34-35)."""
    out = np.zeros(tuple(int(n) for n in Nd), dtype=np.complex128)
    for ci, yi in zip(c, y):
        out += np.conj(ci) * adjoint(yi, om, Nd, Kd, Jd)
    return out


def selfadjoint_coils(x, c, om, Nd, Kd, Jd):
    """A_multi^H A_multi x = sum_i conj(c_i) . A^H A . c_i . x   (eqs. 34-35)."""
    return adjoint_coils(forward_coils(x, c, om, Nd, Kd, Jd), c, om, Nd, Kd, Jd)


# ----------------------------------------------------------------------------------------------------------
# The plain definition the method approximates: the non-uniform DFT (brute force; tiny inputs only)
# ----------------------------------------------------------------------------------------------------------
def _ndft_factors(om, Nd, sign):
    om = np.asarray(om, dtype=np.float64)
    return [np.exp(sign * 1j * om[:, a:a + 1] * (np.arange(N) - N / 2.0)[None, :]) for a, N in enumerate(Nd)]


def ndft_forward(x, om, Nd):
    """(A_exact x)[m] = sum_n x[n] exp(-i sum_a om[m,a] (n_a - N_a/2))."""
    x = np.asarray(x, dtype=np.complex128)
    E = _ndft_factors(om, Nd, -1.0)
    if len(Nd) == 1:
        return np.einsum("ma,a->m", E[0], x)
    if len(Nd) == 2:
        return np.einsum("ma,ab,mb->m", E[0], x, E[1], optimize=True)
    return np.einsum("ma,mb,mc,abc->m", E[0], E[1], E[2], x, optimize=True)


def ndft_adjoint(y, om, Nd):
    """(A_exact^H y)[n] = sum_m y[m] exp(+i sum_a om[m,a] (n_a - N_a/2))."""
    y = np.asarray(y, dtype=np.complex128)
    E = _ndft_factors(om, Nd, +1.0)
    if len(Nd) == 1:
        return np.einsum("m,ma->a", y, E[0])
    if len(Nd) == 2:
        return np.einsum("m,ma,mb->ab", y, E[0], E[1], optimize=True)
    return np.einsum("m,ma,mb,mc->abc", y, E[0], E[1], E[2], optimize=True)
