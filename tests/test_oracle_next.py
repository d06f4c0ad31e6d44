"""Pins of oracle/next_oracle.py (density compensation eqs. (6)-(7), Toeplitz A^H A) against what the mathematics fixes:
closed forms on Cartesian sampling, brute-force sums and the dense non-uniform-DFT matrix on tiny inputs."""
import numpy as np

from oracle import next_oracle as nxt
from oracle import nufft_oracle as orc


def rel(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def cartesian_om(N):
    k = 2 * np.pi * (np.arange(N) - N // 2) / N
    g = np.meshgrid(k, k, indexing="ij")
    return np.stack([g[0].ravel(), g[1].ravel()], axis=1)


def dense_ndft(om, Nd):
    """A_exact[m, n] = exp(-i om_m . (n - N/2)) from the plain definition."""
    axes = [np.arange(n) - n / 2.0 for n in Nd]
    pos = np.stack([g.ravel() for g in np.meshgrid(*axes, indexing="ij")], axis=1)
    return np.exp(-1j * (om @ pos.T))


def test_density_weights_cartesian_closed_form():
    # full Cartesian sampling: A A^H = prod(N) I exactly for the plain DFT, so w = 1/prod(N) after one step and stays
    N = 16
    Nd, Kd, Jd = (N, N), (2 * N, 2 * N), (6, 6)
    om = cartesian_om(N)
    for niter in (1, 3):
        w = nxt.density_weights(om, Nd, Kd, Jd, niter)
        assert np.allclose(w, 1.0 / (N * N), rtol=2e-4)


def test_density_weights_halve_when_every_location_is_duplicated():
    rng = np.random.default_rng(3)
    Nd, Kd, Jd = (12, 12), (24, 24), (6, 6)
    om = rng.uniform(-np.pi, np.pi, (150, 2))
    w1 = nxt.density_weights(om, Nd, Kd, Jd, 4)
    w2 = nxt.density_weights(np.concatenate([om, om]), Nd, Kd, Jd, 4)
    assert np.allclose(w2[:150], 0.5 * w1, rtol=1e-10) and np.allclose(w2[150:], 0.5 * w1, rtol=1e-10)


def test_density_iteration_matches_the_printed_formula_with_the_exact_operator():
    # eq. (6) with A replaced by the dense non-uniform DFT matrix (tiny case): same iteration, kernel error only
    rng = np.random.default_rng(4)
    Nd, Kd, Jd = (8, 8), (16, 16), (6, 6)
    om = rng.uniform(-np.pi, np.pi, (90, 2))
    A = dense_ndft(om, Nd)
    w = np.ones(90)
    for _ in range(3):
        w = w / np.abs(A @ (A.conj().T @ w))
    assert rel(nxt.density_weights(om, Nd, Kd, Jd, 3), w) < 1e-4


def test_adjoint_dcf_inverts_cartesian_sampling():
    N = 16
    Nd, Kd, Jd = (N, N), (2 * N, 2 * N), (6, 6)
    om = cartesian_om(N)
    rng = np.random.default_rng(5)
    x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
    w = nxt.density_weights(om, Nd, Kd, Jd, 1)
    y = orc.forward(x, om, Nd, Kd, Jd)
    assert rel(nxt.adjoint_dcf(y, w, om, Nd, Kd, Jd), x) < 1e-4
    assert np.array_equal(nxt.adjoint_dcf(y, w, om, Nd, Kd, Jd), orc.adjoint(y * w, om, Nd, Kd, Jd))


def test_toeplitz_kernel_against_brute_force_psf():
    rng = np.random.default_rng(6)
    Nd, Kd, Jd = (8, 10), (16, 20), (6, 6)
    om = rng.uniform(-np.pi, np.pi, (200, 2))
    w = rng.uniform(0.5, 1.5, 200)
    _, T = nxt.toeplitz_kernel(om, Nd, Kd, Jd, w)
    d0 = np.arange(-Nd[0], Nd[0])
    d1 = np.arange(-Nd[1], Nd[1])
    exact = np.einsum("m,ma,mb->ab", w, np.exp(1j * np.outer(om[:, 0], d0)), np.exp(1j * np.outer(om[:, 1], d1)))
    exact[0, :] = 0.0
    exact[:, 0] = 0.0
    assert rel(T, exact) < 1e-4
    # Hermitian symmetry T[-d] = conj(T[d]) on the interior |d| <= N-1
    Ti = T[1:, 1:]
    assert np.allclose(Ti[::-1, ::-1], np.conj(Ti), atol=1e-4 * np.abs(T).max())


def test_selfadjoint_toeplitz_against_dense_normal_matrix_and_back_to_back():
    rng = np.random.default_rng(7)
    for Nd in ((8, 8), (6, 12)):
        Kd, Jd = tuple(2 * n for n in Nd), (6, 6)
        om = rng.uniform(-np.pi, np.pi, (300, 2))
        x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
        That, _ = nxt.toeplitz_kernel(om, Nd, Kd, Jd)
        got = nxt.selfadjoint_toeplitz(x, That, Nd)
        A = dense_ndft(om, Nd)
        exact = (A.conj().T @ (A @ x.ravel())).reshape(Nd)
        assert rel(got, exact) < 1e-4
        assert rel(got, orc.selfadjoint(x, om, Nd, Kd, Jd)) < 1e-4


def test_selfadjoint_toeplitz_3d_tiny():
    rng = np.random.default_rng(8)
    Nd, Kd, Jd = (6, 6, 8), (12, 12, 16), (6, 6, 6)
    om = rng.uniform(-np.pi, np.pi, (250, 3))
    x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
    That, _ = nxt.toeplitz_kernel(om, Nd, Kd, Jd)
    A = dense_ndft(om, Nd)
    exact = (A.conj().T @ (A @ x.ravel())).reshape(Nd)
    assert rel(nxt.selfadjoint_toeplitz(x, That, Nd), exact) < 1e-4


# ---- L1TV-LAD: sanity pins (the converged values are pinned in tests/test_oracle_bregman.py) ----
def _lad_problem(seed=11, N=12, M=500):
    from oracle import solvers_oracle as sol  # noqa: F401
    rng = np.random.default_rng(seed)
    Nd, Kd, Jd = (N, N), (2 * N, 2 * N), (6, 6)
    om = rng.uniform(-np.pi, np.pi, (M, 2))
    xt = np.zeros(Nd, dtype=np.complex128)
    xt[3:8, 4:9] = 1.0 + 0.5j
    y = orc.forward(xt, om, Nd, Kd, Jd)
    AHA = lambda z: orc.selfadjoint(z, om, Nd, Kd, Jd)
    return AHA, orc.adjoint(y, om, Nd, Kd, Jd), xt


def test_lad_first_inner_iteration_equals_ols():
    from oracle import solvers_oracle as sol
    AHA, AHy, _ = _lad_problem()
    a = nxt.l1tv_lad(AHA, AHy, 1.0, 0.05, 1, 1, 4)
    b = sol.l1tv_ols(AHA, AHy, 1.0, 0.05, 1, 1, 4)
    assert np.array_equal(a, b)          # d_f = b_f = 0 before the first data-term shrink
    a2 = nxt.l1tv_lad(AHA, AHy, 1.0, 0.05, 1, 3, 4)
    b2 = sol.l1tv_ols(AHA, AHy, 1.0, 0.05, 1, 3, 4)
    assert rel(a2, b2) > 1e-6            # and the data-term split does act afterwards


def test_lad_scale_equivariance_and_progress():
    AHA, AHy, xt = _lad_problem()
    x1 = nxt.l1tv_lad(AHA, AHy, 1.0, 0.05, 2, 3, 4)
    x2 = nxt.l1tv_lad(AHA, 7.5 * AHy, 1.0, 0.05, 2, 3, 4)
    assert rel(x2, 7.5 * x1) < 1e-12
    x0 = nxt.l1tv_lad(AHA, AHy, 1.0, 0.05, 1, 1, 1)
    assert rel(x1, xt) < rel(x0, xt)     # more iterations move towards the piecewise-constant truth


# ---- k-space CG, eqs. (8)-(11) ----
def test_cg_kspace_final_step_inverts_FS():
    rng = np.random.default_rng(12)
    Nd, Kd, Jd = (8, 12), (16, 24), (6, 6)
    x0 = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
    k = orc.scale_pad_fft(x0, Nd, Kd, Jd)
    # zero iterations from a given k: reuse the function's final step through a 0-iteration solve of a trivial problem
    g = np.fft.ifftn(k)
    idx = np.ix_(*[(np.arange(n) - n // 2) % K for n, K in zip(Nd, Kd)])
    x = g[idx] / np.outer(orc.scaling_factors(8, 16, 6), orc.scaling_factors(12, 24, 6))
    assert rel(x, x0) < 1e-13


def test_cg_kspace_converges_to_min_norm_least_squares_of_dense_V():
    rng = np.random.default_rng(13)
    Nd, Kd, Jd = (4, 4), (8, 8), (6, 6)
    om = rng.uniform(-np.pi, np.pi, (40, 2))
    y = rng.standard_normal(40) + 1j * rng.standard_normal(40)
    # dense V from the oracle's own interpolation of unit grids (columns), 40 x 64
    V = np.zeros((40, 64), dtype=np.complex128)
    for j in range(64):
        e = np.zeros(64, dtype=np.complex128)
        e[j] = 1.0
        V[:, j] = orc.interp(e.reshape(Kd), om, Nd, Kd, Jd)
    kls = np.linalg.lstsq(V, y, rcond=None)[0]           # minimum-norm least-squares solution
    x, k = nxt.cg_kspace(y, om, Nd, Kd, Jd, 100)      # kappa(V)^2 ~ 1.4e4: ~100 iterations to converge in float64
    assert rel(k.ravel(), kls) < 1e-8
    # and x is S^-1 F^-1 of that k
    g = np.fft.ifftn(kls.reshape(Kd))
    idx = np.ix_(*[(np.arange(n) - n // 2) % K for n, K in zip(Nd, Kd)])
    xr = g[idx] / np.outer(orc.scaling_factors(4, 8, 6), orc.scaling_factors(4, 8, 6))
    assert rel(x, xr) < 1e-8
