"""Mathematical pins of the split-Bregman oracles (oracle/solvers_oracle.py:l1tv_ols, oracle/next_oracle.py:l1tv_lad).

The paper prints no iterate values (eqs. (13)-(22), :204-249 eqs. (23)-(33)), so these pins come from
what the iterations must converge to, computed WITHOUT the oracle's formulas:

  * Cartesian full sampling makes A^H A = prod(N) I.  With one outer iteration and many inner ones, L1TV-OLS is then
    anisotropic TV denoising, whose minimiser for a two-level image (a box of L rows on a periodic axis) is known in
    closed form: the plateaus move towards each other by 2/(kappa L) and 2/(kappa (N - L)) (kappa = data weight).  The
    result must not depend on lambda (a penalty parameter of the splitting): a shrink threshold lambda instead of
    1/lambda, or a flipped sign in a Bregman update, breaks this.
  * The outer update, eq. (22) / (33), is a Bregman iteration on the data term: with it the iterates converge to the
    data-consistent solution A^H A x = A^H y (here x = z exactly); without it they stay at the denoised image.
  * On a small NON-Cartesian problem the converged L1TV-OLS result must be the minimiser of
    mu/2 ||A x - y||^2 + w (||grad_0 x||_1 + ||grad_1 x||_1), w = max|A^H y| (the oracle's scaling, reading R17); that
    minimiser is computed here by a different algorithm (Chambolle-Pock primal-dual iterations on dense matrices).
  * L1TV-LAD with A^H A = P I converges to the minimiser of ||x - z||_1 + TV(x) (TV-L1 denoising), which is contrast
    invariant: a box wider than 2 rows keeps its full height, a one-row line is removed entirely -- for every mu, lambda.
    A threshold mu instead of 1/mu (or lambda instead of 1/lambda) moves the keep / remove boundary and fails.
"""
import numpy as np

import workloads as wl
from oracle import next_oracle as nxt
from oracle import solvers_oracle as sol

N0, N1, L = 16, 8, 6
P = N0 * N1
PHASE = np.exp(0.7j)


def box_image(h=2.0):
    z = np.zeros((N0, N1), dtype=np.complex128)
    z[3:3 + L, :] = h * PHASE
    return z


def test_l1tv_ols_cartesian_box_has_the_tv_denoising_closed_form_for_every_lambda():
    h, mu = 2.0, 2.0
    z = box_image(h)
    inside = (np.arange(N0) >= 3) & (np.arange(N0) < 3 + L)
    # returned image = argmin mu/2 P ||x - z||^2 ... in the oracle's scaling: a = h (1 - 2/(mu L)), b = 2 h / (mu (N0 - L))
    a, b = h * (1.0 - 2.0 / (mu * L)), 2.0 * h / (mu * (N0 - L))
    expect = PHASE * np.where(inside[:, None], a, b) * np.ones((1, N1))
    for lam in (100.0, 1000.0):
        x = sol.l1tv_ols(lambda v: P * v, P * z, mu, lam, 1, 400, 30)
        assert np.abs(x - expect).max() < 1e-10, (lam, np.abs(x - expect).max())
    # the plateau values are not those of the data: the pin has teeth
    assert abs(a - h) > 0.3 and b > 0.15


def test_l1tv_ols_outer_bregman_iterations_converge_to_the_data_consistent_image():
    z = box_image()
    one = sol.l1tv_ols(lambda v: P * v, P * z, 2.0, 100.0, 1, 30, 30)
    many = sol.l1tv_ols(lambda v: P * v, P * z, 2.0, 100.0, 10, 30, 30)
    assert np.linalg.norm(one - z) / np.linalg.norm(z) > 0.15        # one group of inner iterations: the denoised image
    assert np.linalg.norm(many - z) / np.linalg.norm(z) < 1e-9       # eq. (22) adds the residual back: x -> z


def _dense_problem():
    Nd = (8, 8)
    om = wl.traj_uniform(160, 2, seed=71)
    cols = np.stack(np.meshgrid(np.arange(8) - 4.0, np.arange(8) - 4.0, indexing="ij"), axis=-1).reshape(-1, 2)
    A = np.exp(-1j * (om @ cols.T))                                  # plain non-uniform DFT matrix, 160 x 64
    rng = np.random.default_rng(72)
    truth = np.zeros(Nd)
    truth[2:6, 1:5] = 1.0
    truth[4:7, 5:7] = -0.5
    y = A @ truth.ravel() + 0.3 * (rng.standard_normal(160) + 1j * rng.standard_normal(160))
    return Nd, A, y


def _grad_matrix(Nd, axis):
    n = Nd[0] * Nd[1]
    G = np.zeros((n, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1.0
        G[:, j] = (np.roll(e.reshape(Nd), -1, axis=axis) - e.reshape(Nd)).ravel()      # eq. (12), periodic (R15)
    return G


def test_l1tv_ols_converges_to_the_minimiser_found_by_a_primal_dual_method():
    Nd, A, y = _dense_problem()
    mu = 0.05
    AHA = A.conj().T @ A
    AHy = A.conj().T @ y
    w = np.max(np.abs(AHy))                                          # TV weight of the unscaled problem (R17)
    x_sb = sol.l1tv_ols(lambda v: (AHA @ v.ravel()).reshape(Nd), AHy.reshape(Nd), mu, 4.0, 1, 3000, 70).ravel()
    # Chambolle-Pock on  min_x mu/2 ||A x - y||^2 + w ||K x||_1,  K = [grad_0; grad_1]
    K = np.vstack([_grad_matrix(Nd, 0), _grad_matrix(Nd, 1)])
    tau = sigma = 0.33                                               # tau sigma ||K||^2 <= 0.33^2 * 8 < 1
    Minv = np.linalg.inv(np.eye(64) + tau * mu * AHA)
    x = np.zeros(64, dtype=np.complex128)
    xb = x.copy()
    p = np.zeros(128, dtype=np.complex128)
    for _ in range(60000):
        p = p + sigma * (K @ xb)
        p = p * (w / np.maximum(np.abs(p), w))                        # projection onto |p| <= w
        xn = Minv @ (x - tau * (K.T @ p) + tau * mu * AHy)
        xb = 2.0 * xn - x
        x = xn

    def objective(v):
        return 0.5 * mu * np.linalg.norm(A @ v - y) ** 2 + w * np.abs(K @ v).sum()

    assert np.linalg.norm(x_sb - x) / np.linalg.norm(x) < 2e-4
    assert objective(x_sb) <= objective(x) * (1.0 + 1e-7)
    # and it is a genuinely regularised solution, not least squares
    x_ls = np.linalg.lstsq(A, y, rcond=None)[0]
    assert np.linalg.norm(x_sb - x_ls) / np.linalg.norm(x_ls) > 0.05


def lad_image():
    z = box_image(2.0)
    z[12, :] = 1.5 * PHASE                                           # one-row line
    return z


def test_l1tv_lad_cartesian_is_contrast_invariant_tv_l1_denoising_for_every_mu_lambda():
    z = lad_image()
    for mu, lam in ((2.0, 4.0), (0.5, 3.0)):
        x = nxt.l1tv_lad(lambda v: P * v, P * z, mu, lam, 1, 1500, 30)
        assert np.abs(x[3:3 + L, :] - 2.0 * PHASE).max() < 1e-8     # wide box (L = 6 > 2): kept at FULL height
        assert np.abs(x[12, :]).max() < 1e-5                         # one-row line (1 < 2): removed
        assert np.abs(x[0, :]).max() < 1e-8
    # L1TV-OLS on the same data loses contrast (its box is h (1 - 2/(mu L))): the two solvers are told apart
    xo = sol.l1tv_ols(lambda v: P * v, P * z, 2.0, 100.0, 1, 400, 30)
    assert abs(abs(xo[5, 3]) - 2.0) > 0.2


def test_l1tv_lad_outer_bregman_iterations_restore_the_removed_line():
    z = lad_image()
    one = nxt.l1tv_lad(lambda v: P * v, P * z, 1.0, 2.0, 1, 30, 30)
    many = nxt.l1tv_lad(lambda v: P * v, P * z, 1.0, 2.0, 10, 30, 30)
    assert abs(abs(one[12, 3]) - 1.5) > 0.02                         # already shrinking after one group of 30
    assert np.linalg.norm(many - z) / np.linalg.norm(z) < 1e-9       # eq. (33): x -> z, line restored
