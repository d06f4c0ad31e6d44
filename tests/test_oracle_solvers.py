"""Pins for oracle/solvers_oracle.py: gradient, shrink, CG, and sanity pins of L1TV-OLS (its converged values: test_oracle_bregman.py)."""
import numpy as np
import pytest

import workloads as wl
from oracle import nufft_oracle as orc
from oracle import solvers_oracle as sol


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def test_gradient_closed_form_and_exact_adjoint():
    x = np.arange(20.0).reshape(4, 5) ** 2 + 1j * np.arange(20.0).reshape(4, 5)
    g0 = sol.grad(x, 0)
    assert g0[1, 2] == x[2, 2] - x[1, 2]            # eq. (12)
    assert g0[3, 2] == x[0, 2] - x[3, 2]            # periodic (reading R15)
    g1 = sol.grad(x, 1)
    assert g1[2, 4] == x[2, 0] - x[2, 4]
    rng = np.random.default_rng(0)
    x = rng.standard_normal((6, 7)) + 1j * rng.standard_normal((6, 7))
    d = rng.standard_normal((6, 7)) + 1j * rng.standard_normal((6, 7))
    for a in (0, 1):
        assert abs(np.vdot(sol.grad(x, a), d) - np.vdot(x, sol.grad_T(d, a))) < 1e-12
        # dense matrix of grad and its transpose
        n = x.size
        Gm = np.zeros((n, n))
        for j in range(n):
            e = np.zeros(n)
            e[j] = 1
            Gm[:, j] = sol.grad(e.reshape(6, 7), a).ravel().real
        assert np.allclose(Gm.T @ d.ravel(), sol.grad_T(d, a).ravel())


def test_shrink_closed_form():
    z = np.array([3 + 4j, 0.0, -0.5j, 2.0, -10.0])
    out = sol.shrink(z, 1.0)
    assert out[0] == pytest.approx((3 + 4j) * 4 / 5)
    assert out[1] == 0 and out[2] == 0
    assert out[3] == pytest.approx(1.0) and out[4] == pytest.approx(-9.0)
    rng = np.random.default_rng(1)
    z = rng.standard_normal(100) + 1j * rng.standard_normal(100)
    s = sol.shrink(z, 0.7)
    assert np.allclose(np.abs(s), np.maximum(np.abs(z) - 0.7, 0))
    nz = np.abs(s) > 0
    assert np.allclose(np.angle(s[nz]), np.angle(z[nz]))
    assert np.all(sol.shrink(z, np.inf) == 0)
    assert np.allclose(sol.shrink(z, 0.0), z)


def test_cg_iterates_are_krylov_minimisers_and_converge_to_lstsq():
    """Tiny dense problem: A = dense NDFT matrix; CG iterate k minimises the A^H A-norm of the error
    over span{b, Tb, .., T^{k-1} b}; the converged iterate equals lstsq."""
    Nd = (6, 6)
    om = wl.traj_uniform(200, 2, seed=61)
    cols = np.stack(np.meshgrid(np.arange(6) - 3.0, np.arange(6) - 3.0, indexing="ij"), axis=-1).reshape(-1, 2)
    A = np.exp(-1j * (om @ cols.T))
    rng = np.random.default_rng(62)
    y = rng.standard_normal(200) + 1j * rng.standard_normal(200)
    T = A.conj().T @ A
    b = A.conj().T @ y
    xs = np.linalg.lstsq(A, y, rcond=None)[0]
    x, hist = sol.cg(lambda v: (T @ v.ravel()).reshape(Nd), b.reshape(Nd), 36)
    assert rel(x.ravel(), xs) < 1e-10
    assert hist[0] == pytest.approx(np.linalg.norm(b)) and hist[-1] < 1e-9 * hist[0]
    for k in (1, 2, 5):
        xk, hk = sol.cg(lambda v: (T @ v.ravel()).reshape(Nd), b.reshape(Nd), k)
        Kry = np.stack([np.linalg.matrix_power(T, j) @ b for j in range(k)], axis=1)
        # minimise (x - xs)^H T (x - xs) over x = Kry c   ->  (Kry^H T Kry) c = Kry^H b
        c = np.linalg.solve(Kry.conj().T @ T @ Kry, Kry.conj().T @ b)
        assert rel(xk.ravel(), Kry @ c) < 1e-8
        assert hk[-1] == pytest.approx(np.linalg.norm(b - T @ xk.ravel()), rel=1e-8)


def test_cg_with_oracle_nufft_operator_reduces_residual():
    cfg = wl.config(0, 4)
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    x_true = wl.image_gaussian(Nd, seed=63).astype(np.complex128)
    y = orc.forward(x_true, om, Nd, Kd, Jd)
    AHA = lambda v: orc.selfadjoint(v, om, Nd, Kd, Jd)
    x, hist = sol.cg(AHA, orc.adjoint(y, om, Nd, Kd, Jd), 120)
    assert hist[-1] < 1e-10 * hist[0]
    assert rel(x, x_true) < 1e-9          # consistent data, 2x oversampled uniform sampling: recovers x exactly


def _setup_l1(seed=70):
    cfg = wl.config(4, 16)                # 16 x 16 image, 8 spokes x 32, 8 coils
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    c = wl.coil_maps(4, Nd).astype(np.complex128)
    ph = wl.phantom(Nd).astype(np.complex128)
    y = orc.forward_coils(ph, c, om, Nd, Kd, Jd)
    y = y + wl.noise_like(y)
    AHA = lambda v: orc.selfadjoint_coils(v, c, om, Nd, Kd, Jd)
    AHy = orc.adjoint_coils(y, c, om, Nd, Kd, Jd)
    return AHA, AHy, ph


def test_l1tv_lambda_zero_single_outer_is_cg_on_normal_equation():
    """lambda = 0, one outer, one inner iteration: rhs = mu A^H y, K = mu A^H A -> n_cg steps of CG (x0 = 0) on the
    normal equation; scaling by max|A^H y| (R17) must cancel."""
    AHA, AHy, _ = _setup_l1()
    x = sol.l1tv_ols(AHA, AHy, mu=1.0, lam=0.0, n_outer=1, n_inner=1, n_cg=7)
    xc, _ = sol.cg(AHA, AHy, 7)
    assert rel(x, xc) < 1e-11
    x2 = sol.l1tv_ols(AHA, AHy, mu=3.0, lam=0.0, n_outer=1, n_inner=1, n_cg=7)
    assert rel(x2, xc) < 1e-11            # mu cancels when lambda = 0


def test_l1tv_shrink_active_and_scale_equivariance():
    AHA, AHy, ph = _setup_l1()
    gain = np.max(np.abs(AHA(np.ones_like(AHy))))
    lam = 5.0 * gain                       # threshold 1/lambda comparable with |grad x| of the scaled problem
    x, trace = sol.l1tv_ols(AHA, AHy, mu=1.0, lam=lam, n_outer=2, n_inner=3, n_cg=3, return_trace=True)
    assert len(trace) == 6 and np.all(np.isfinite(x))
    x0 = sol.l1tv_ols(AHA, AHy, mu=1.0, lam=0.0, n_outer=2, n_inner=3, n_cg=3)
    assert rel(x, x0) > 1e-3               # regularisation does something
    tv = lambda v: np.sum(np.abs(sol.grad(v, 0))) + np.sum(np.abs(sol.grad(v, 1)))
    assert tv(x) < tv(x0)                  # and it lowers the total variation
    # R17: the result is equivariant to scaling y
    xs = sol.l1tv_ols(AHA, 7.5 * AHy, mu=1.0, lam=lam, n_outer=2, n_inner=3, n_cg=3)
    assert rel(xs, 7.5 * x) < 1e-10
