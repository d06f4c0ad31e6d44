"""Float64 CPU oracle of the rows SURVEY.md 8(f) marks "next".   TEST INFRASTRUCTURE.

    density_weights / adjoint_dcf   sampling density compensation, eqs. (6)-(7)
    toeplitz_kernel / selfadjoint_toeplitz   "precomputing A^H A" (Toeplitz, ref. [6])   PAPER.md:86-98, Fig. 3 :114
    l1tv_lad                        split-Bregman L1TV-LAD, eqs. (23)-(33)
    cg_kspace                       the paper's k-space CG  V^H V k = V^H y, x = S^-1 F^-1 k   PAPER.md:124-143, eqs. (8)-(11)

Built on oracle/nufft_oracle.py (forward, adjoint); numpy float64 / complex128; numpy.fft as a library step.

Readings of the paper taken here (R21-R24; R23 and R24 are stated in the docstrings of l1tv_lad and cg_kspace):
    R21  eq. (6) w_{i+1} = w_i / (A A^H w_i): the paper gives neither w_0, nor the iteration count, nor how a complex
         A A^H w is divided into a real density function.  Taken: w_0 = 1, w real, w_{i+1} = w_i / |A A^H w_i|
         (elementwise magnitude, as in ref. [7]'s iteration), a fixed iteration count given by the caller.
    R22  the paper's own "Toeplitz" precomputes the sparse V^H V; SURVEY 8(f)-1 asks for the true
         Toeplitz embedding of ref. [6]: A^H A x = crop(F^H(T^ . F(pad x))) on the 2N grid, T^ = F(T),
         T[d] = sum_m w_m e^{i om_m . d}, d in [-N, N)^dim, obtained from 2^dim adjoint NUFFTs of phase-modulated weights
         on the plan's own geometry (one per half-shift s in {-N/2, +N/2}^dim; no larger grid is needed, so every
         supported size works).  It equals the back-to-back operator up to the interpolation-kernel error (~1e-5), not
         to rounding.

Parity pins (tests/test_oracle_next.py):
    density_weights        Cartesian full sampling: fixed point w = 1 / prod(N) (closed form, A A^H = prod(N) I);
                           every location duplicated: the weights halve; invariance to the scale of w_0 after one step
    adjoint_dcf            = adjoint(y * w) by definition; Cartesian case inverts the DFT: A^H(w . A x) = x
    toeplitz_kernel        T[d] against the brute-force sum over samples on tiny sizes (rel. <= 1e-4); Hermitian symmetry
                           T[-d] = conj(T[d])
    selfadjoint_toeplitz   against the dense matrix A_exact^H A_exact built from the plain non-uniform DFT definition
                           (rel. <= 1e-4) and against adjoint(forward(x)) (same bound)
    l1tv_lad               tests/test_oracle_bregman.py: with A^H A = prod(N) I the converged result is TV-L1 denoising,
                           contrast invariant for every mu, lambda: a box wider than two rows keeps its full height, a
                           one-row line is removed; the outer update eq. (33) restores the line (x -> z).  A threshold mu
                           for 1/mu (or lambda for 1/lambda), a flipped b_f update or a dropped eq. (33) each fail.  Also:
                           first inner iteration = L1TV-OLS's, scale equivariance, consistent-data fixed point.
    cg_kspace              final step: S^{-1}F^{-1} inverts k = F S x exactly; converged k equals the minimum-norm least
                           squares solution pinv(V) y computed from the dense V (numpy.linalg.lstsq); CG recurrence itself
                           pinned in tests/test_oracle_solvers.py
No function here is "parity unpinned".
"""
import numpy as np

from . import nufft_oracle as orc

__all__ = ["density_weights", "adjoint_dcf", "toeplitz_kernel", "selfadjoint_toeplitz", "l1tv_lad", "cg_kspace"]


def density_weights(om, Nd, Kd, Jd, niter):
    """Sampling density compensation function, eq. (6) PAPER.md:118 with reading R21:
    w_0 = 1;  w_{i+1} = w_i / |A A^H w_i|.   Returns real float64 w[M]."""
    M = np.asarray(om).shape[0]
    w = np.ones(M, dtype=np.float64)
    for _ in range(int(niter)):
        t = orc.forward(orc.adjoint(w.astype(np.complex128), om, Nd, Kd, Jd), om, Nd, Kd, Jd)
        w = w / np.abs(t)
    return w


def adjoint_dcf(y, w, om, Nd, Kd, Jd):
    """x = A^H (y . w), eq. (7) PAPER.md:122."""
    return orc.adjoint(np.asarray(y, dtype=np.complex128) * np.asarray(w), om, Nd, Kd, Jd)


def toeplitz_kernel(om, Nd, Kd, Jd, w=None):
    """T^ = FFT over the 2N grid of the point-spread function T[d] = sum_m w_m e^{i om_m . d}, d in [-N, N)^dim (R22).
    T is assembled from 2^dim adjoint NUFFTs on the SAME Nd / Kd geometry: with d = d' + s, d' in [-N/2, N/2)^dim and
    s in {-N/2, +N/2}^dim,  T[d' + s] = sum_m (w_m e^{i om_m . s}) e^{i om_m . d'}  is the adjoint NUFFT of the modulated
    weights, whose pixel n sits at position n - N/2 = d'.  Block h in {0,1}^dim (s_a = (h_a - 1/2) N_a) fills
    T[h_a N_a : (h_a + 1) N_a] of the array indexed by n2 = d + N.  Returns (T^ complex128 of shape 2N, T)."""
    import itertools
    Nd = tuple(int(n) for n in Nd)
    om = np.asarray(om, dtype=np.float64)
    M = om.shape[0]
    wv = np.ones(M, dtype=np.complex128) if w is None else np.asarray(w, dtype=np.complex128)
    T = np.zeros(tuple(2 * n for n in Nd), dtype=np.complex128)
    for h in itertools.product((0, 1), repeat=len(Nd)):
        shift = np.array([(ha - 0.5) * n for ha, n in zip(h, Nd)])
        blk = orc.adjoint(wv * np.exp(1j * (om @ shift)), om, Nd, Kd, Jd)
        T[tuple(slice(ha * n, (ha + 1) * n) for ha, n in zip(h, Nd))] = blk
    # d = -N (pixel 0 on every axis) is never used by a linear convolution of two length-N supports; drop it
    for a in range(len(Nd)):
        sl = [slice(None)] * len(Nd)
        sl[a] = 0
        T[tuple(sl)] = 0.0
    That = np.fft.fftn(np.fft.ifftshift(T))          # index d mod 2N
    return That, T


def selfadjoint_toeplitz(x, That, Nd):
    """A^H A x by Toeplitz embedding (R22): zero-pad x to 2N, multiply the spectra, crop.
    (T * x)[n] = sum_n' T[n - n'] x[n'] for n in [0, N): the circular convolution of size 2N is alias-free."""
    Nd = tuple(int(n) for n in Nd)
    z = np.zeros(That.shape, dtype=np.complex128)
    z[tuple(slice(0, n) for n in Nd)] = x
    r = np.fft.ifftn(np.fft.fftn(z) * That)
    return r[tuple(slice(0, n) for n in Nd)]


def l1tv_lad(AHA, AHy, mu, lam, n_outer, n_inner, n_cg):
    """Split-Bregman L1TV-LAD, eqs. (23)-(33), with the readings of L1TV-OLS (R13-R18: two gradient
    splits, complex soft threshold, periodic gradient, n_cg warm-started CG steps for eq. (26), scaling by
    1/max|A^H y|) and, for the data-term split (R23): eq. (29) prints `b_y^k` where the pattern of eqs. (25), (32)
    requires b_f^k; the `A^H y` of eqs. (29) and (32) is the (scaled) A^H y itself, not the Bregman-updated A^H y^k:
        rhs  = mu (A^H y^k + d_f - b_f) + lam sum_a grad_a^T (d_a - b_a)                      (25)
        x    = K^{-1} rhs,   K = mu A^H A + lam sum_a grad_a^T grad_a                          (24), (26)
        d_a  = shrink(grad_a x + b_a, 1/lam);   b_a += grad_a x - d_a                         (27)-(28), (30)-(31)
        r    = A^H A x - A^H y;   d_f = shrink(r + b_f, 1/mu);   b_f += r - d_f               (29), (32)
        outer: A^H y^{k+1} = A^H y^k + A^H y - A^H A x                                        (33)
    Pins: tests/test_oracle_bregman.py (converged values in closed form on Cartesian sampling, outer update) and
    tests/test_oracle_next.py (first inner iteration equals L1TV-OLS's, scale equivariance, consistent-data fixed point)."""
    from .solvers_oracle import cg_steps, grad, grad_T, shrink
    AHy = np.asarray(AHy, dtype=np.complex128)
    assert AHy.ndim == 2
    c = 1.0 / np.max(np.abs(AHy))
    AHy_s = AHy * c
    AHy_k = AHy_s.copy()
    x = np.zeros_like(AHy_s)
    d = [np.zeros_like(AHy_s) for _ in range(2)]
    b = [np.zeros_like(AHy_s) for _ in range(2)]
    d_f = np.zeros_like(AHy_s)
    b_f = np.zeros_like(AHy_s)

    def K(z):                                         # eq. (24)
        out = mu * AHA(z)
        for a in range(2):
            out = out + lam * grad_T(grad(z, a), a)
        return out

    thr = 1.0 / lam if lam > 0.0 else np.inf
    thr_f = 1.0 / mu if mu > 0.0 else np.inf
    for _ in range(int(n_outer)):
        for _ in range(int(n_inner)):
            rhs = mu * (AHy_k + d_f - b_f)            # eq. (25)
            for a in range(2):
                rhs = rhs + lam * grad_T(d[a] - b[a], a)
            x, _ = cg_steps(K, rhs, x, n_cg)          # eq. (26)
            for a in range(2):
                g = grad(x, a)
                d[a] = shrink(g + b[a], thr)          # eqs. (27)-(28)
                b[a] = b[a] + (g - d[a])              # eqs. (30)-(31)
            r = AHA(x) - AHy_s
            d_f = shrink(r + b_f, thr_f)              # eq. (29)
            b_f = b_f + (r - d_f)                     # eq. (32)
        AHy_k = AHy_k + AHy_s - AHA(x)                # eq. (33)
    return x / c


def cg_kspace(y, om, Nd, Kd, Jd, niter):
    """The paper's own two-step conjugate-gradient solution, eqs. (8)-(11):
        solve  V^H V k = V^H y  for the oversampled grid k by conjugate gradient             (9), (11)
        x = S^{-1} F^{-1} k: inverse FFT, crop, divide by the scaling factor               (10)
    Reading R24: k_0 = 0, exactly niter iterations of linear CG (the same recurrence as solvers_oracle.cg_steps), F^{-1}
    is the normalised inverse DFT (the inverse of F, not its adjoint), the image is read from the circular positions
    (n - N/2) mod K where S placed it (R4).  Returns (x, k)."""
    from .solvers_oracle import cg_steps
    Nd = tuple(int(n) for n in Nd)
    Kd = tuple(int(k) for k in Kd)
    op = lambda g: orc.grid_adjoint(orc.interp(g, om, Nd, Kd, Jd), om, Nd, Kd, Jd)
    rhs = orc.grid_adjoint(np.asarray(y, dtype=np.complex128), om, Nd, Kd, Jd)
    k, _ = cg_steps(op, rhs, np.zeros(Kd, dtype=np.complex128), niter)
    g = np.fft.ifftn(k)                                                   # F^{-1}
    idx = np.ix_(*[(np.arange(n) - n // 2) % K for n, K in zip(Nd, Kd)])   # crop at (n - N/2) mod K
    x = g[idx]
    for a, (n, K, J) in enumerate(zip(Nd, Kd, Jd)):                        # S^{-1}
        shape = [1] * len(Nd)
        shape[a] = n
        x = x / orc.scaling_factors(n, K, J).reshape(shape)
    return x, k
