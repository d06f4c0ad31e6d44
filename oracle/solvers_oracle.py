"""Float64 CPU oracle of the solvers built on A^H A.   TEST INFRASTRUCTURE.

Follows PAPER.md (arxiv 1710.03197) section 2.2, in the paper's order and notation:
    grad / grad_T    image gradient, eq. (12)
    shrink           shrinkage function of eqs. (18)-(19), (29)
    cg               conjugate gradient on the normal equation     PAPER.md:96 (eq. 5), 130-143
    l1tv_ols         split-Bregman L1TV-OLS, eqs. (13)-(22)
The operators are passed in as callables, so this module contains no NUFFT arithmetic of its own.

Readings of the paper taken here (R12-R18):
    R12  CG is linear CG on A^H A x = A^H y (BASELINE config 3), x0 = 0, fixed iteration count, no
         preconditioner; alpha = <r,r> / Re<p, A^H A p>.
    R13  eqs. (18)-(21) are printed twice and garbled; exactly two splits (image axes 0 and 1) are used:
         d_a = shrink(grad_a x + b_a, 1/lambda),  b_a += grad_a x - d_a.
    R14  shrink(z, t) = z * max(|z| - t, 0) / |z| (complex soft threshold), 0 at z = 0; anisotropic.
    R15  grad_a x = roll(x, -1, a) - x (periodic forward difference); grad_a^T d = roll(d, +1, a) - d.
    R16  x = K^{-1} rhs (eq. 17) is n_cg steps of CG on K x = rhs warm-started at the previous x,
         K = mu A^H A + lambda sum_a grad_a^T grad_a (eq. 15).
    R17  y is scaled so that max |A^H y| = 1 before iterating; the result is scaled back.
    R18  the iterations (16)-(22) define the method; eq. (13)'s unsquared norm is not used.

Parity pins (tests/test_oracle_solvers.py):
    grad / grad_T   exact adjoint identity <grad x, d> = <x, grad_T d>; closed form on a ramp
    shrink          closed-form values; magnitude / phase properties
    cg              tiny dense problem: iterate k equals the minimiser of the A-norm error over the k-th Krylov
                    space (computed by dense linear algebra) and converges to numpy.linalg.lstsq
    l1tv_ols        tests/test_oracle_bregman.py: (i) Cartesian full sampling (A^H A = prod(N) I): the converged result is
                    the closed-form TV-denoising minimiser of a two-level image, for every lambda; (ii) the outer
                    update eq. (22) drives the iterates to the data-consistent image; (iii) on a small non-Cartesian
                    dense problem the converged result equals the minimiser of mu/2 ||Ax - y||^2 + w TV(x) computed
                    by Chambolle-Pock primal-dual iterations.  A threshold lambda instead of 1/lambda, a flipped
                    Bregman update or a dropped eq. (22) each fail one of them.  Also: lambda = 0 reduces to CG.
"""
import numpy as np

__all__ = ["grad", "grad_T", "shrink", "cg", "cg_steps", "l1tv_ols", "vdot"]


def vdot(a, b):
    """<a, b> = sum conj(a) b."""
    return np.vdot(np.asarray(a).ravel(), np.asarray(b).ravel())


def grad(x, axis):
    """grad_a x = x(.., a+1, ..) - x(.., a, ..), periodic  (eq. 12; reading R15)."""
    return np.roll(x, -1, axis=axis) - x


def grad_T(d, axis):
    """Exact transpose of grad: grad_a^T d = roll(d, +1, a) - d  (reading R15)."""
    return np.roll(d, 1, axis=axis) - d


def shrink(z, t):
    """Complex soft threshold: z * max(|z| - t, 0) / |z|, and 0 where z = 0  (reading R14)."""
    z = np.asarray(z, dtype=np.complex128)
    mag = np.abs(z)
    safe = np.where(mag > 0.0, mag, 1.0)
    return z * (np.maximum(mag - t, 0.0) / safe)


def cg_steps(op, rhs, x0, niter):
    """niter steps of linear conjugate gradient on op(x) = rhs from x0 (op Hermitian positive semi-definite).

    Returns (x, history) with history[k] = ||r_k||_2 for k = 0..niter.
    """
    x = np.array(x0, dtype=np.complex128, copy=True)
    r = np.asarray(rhs, dtype=np.complex128) - op(x)
    p = r.copy()
    rs = vdot(r, r).real
    hist = [np.sqrt(rs)]
    for _ in range(int(niter)):
        if rs == 0.0:
            hist.append(0.0)
            continue
        Ap = op(p)
        alpha = rs / vdot(p, Ap).real
        x = x + alpha * p
        r = r - alpha * Ap
        rs_new = vdot(r, r).real
        p = r + (rs_new / rs) * p
        rs = rs_new
        hist.append(np.sqrt(rs))
    return x, np.array(hist)


def cg(AHA, AHy, niter):
    """CG on the normal equation A^H A x = A^H y (eq. 5), x0 = 0, fixed niter (reading R12).

    AHA: callable x -> A^H A x;  AHy: the right-hand side A^H y (array of image shape).
    """
    return cg_steps(AHA, AHy, np.zeros_like(np.asarray(AHy, dtype=np.complex128)), niter)


def l1tv_ols(AHA, AHy, mu, lam, n_outer, n_inner, n_cg, return_trace=False):
    """Split-Bregman L1TV-OLS, eqs. (15)-(22), readings R13-R18.

    AHA: callable x -> A^H A x (single- or multi-coil, eq. 34-35);  AHy = A^H y (image shape, 2-D).
    The problem is scaled by c = 1 / max|A^H y| (R17) and the result scaled back.
    """
    AHy = np.asarray(AHy, dtype=np.complex128)
    assert AHy.ndim == 2
    c = 1.0 / np.max(np.abs(AHy))
    AHy_s = AHy * c                                   # A^H y of the scaled problem
    AHy_k = AHy_s.copy()                              # A^H y^k of eq. (22)
    x = np.zeros_like(AHy_s)
    d = [np.zeros_like(AHy_s) for _ in range(2)]
    b = [np.zeros_like(AHy_s) for _ in range(2)]

    def K(z):                                         # eq. (15)
        out = mu * AHA(z)
        for a in range(2):
            out = out + lam * grad_T(grad(z, a), a)
        return out

    thr = 1.0 / lam if lam > 0.0 else np.inf        # shrink threshold 1/lambda
    trace = []
    for _ in range(int(n_outer)):
        for _ in range(int(n_inner)):
            rhs = mu * AHy_k                          # eq. (16)
            for a in range(2):
                rhs = rhs + lam * grad_T(d[a] - b[a], a)
            x, _ = cg_steps(K, rhs, x, n_cg)          # eq. (17), reading R16
            for a in range(2):
                g = grad(x, a)
                d[a] = shrink(g + b[a], thr)          # eqs. (18)-(19)
                b[a] = b[a] + (g - d[a])              # eqs. (20)-(21)
            trace.append(x / c)
        AHy_k = AHy_k + AHy_s - AHA(x)                # eq. (22)
    x = x / c
    return (x, trace) if return_trace else x
