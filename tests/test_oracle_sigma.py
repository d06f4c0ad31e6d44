"""Pins for the oracle at oversampling ratios other than 2 (SURVEY 8(f)-4 "other sigma"; 8(c) reading R2: beta depends on
sigma = K/N "so other Kd/Nd ratios keep working").

Expected values come from the plain definition (dense NDFT matrix built here) and from the aliasing ratio
|Phi(1 - xi_e)| / Phi(xi_e) at the image edge xi_e = N / 2K = 1 / (2 sigma), with Phi obtained by QUADRATURE of the defining
integral and I0 from its power series (not the oracle's closed form): the error of the method must sit within a small
factor of that ratio on both sides, for every sigma -- a beta that ignored sigma, scaling factors evaluated at n/N instead
of n/K, or an image placed at the wrong grid offset all break it.
"""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import nufft_oracle as orc


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def ndft_matrix(om, Nd):
    M, d = om.shape
    cols = np.stack(np.meshgrid(*[np.arange(N) - N / 2.0 for N in Nd], indexing="ij"), axis=-1).reshape(-1, d)
    return np.exp(-1j * (om @ cols.T))


def i0_float(x):
    q, s, term, k = 0.25 * x * x, 0.0, 1.0, 0
    while term > 1e-18 * s:
        s += term
        k += 1
        term *= q / (k * k)
    return s


def Phi_quadrature(xi, J, beta):
    i0b = i0_float(beta)
    f = lambda t: i0_float(beta * math.sqrt(max(0.0, 1.0 - (2.0 * t / J) ** 2))) / i0b
    val, _ = integrate.quad(lambda t: f(t) * math.cos(2 * math.pi * xi * t), -J / 2.0, J / 2.0, limit=200,
                            epsabs=1e-13, epsrel=1e-12)
    return val


CASES = [((20, 40), (32, 64)), ((48, 48), (64, 64)), ((16, 16), (64, 64)), ((12, 12), (32, 32)), ((40,), (64,)),
         ((28, 28), (32, 32)), ((12, 12, 12), (16, 16, 16))]


@pytest.mark.parametrize("Nd,Kd", CASES)
@pytest.mark.parametrize("J", [4, 6])
def test_forward_adjoint_vs_ndft_at_sigma(Nd, Kd, J):
    rng = np.random.default_rng(11)
    d = len(Nd)
    Jd = (J,) * d
    sigma = Kd[0] / Nd[0]
    beta = orc.kb_beta(J, sigma)
    assert beta == pytest.approx(math.pi * math.sqrt((J / sigma) ** 2 * (sigma - 0.5) ** 2 - 0.8), rel=1e-14)
    om = rng.uniform(-np.pi, np.pi, (300, d))
    x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
    y = rng.standard_normal(300) + 1j * rng.standard_normal(300)
    A = ndft_matrix(om, Nd)
    xe = 1.0 / (2.0 * sigma)
    alias = abs(Phi_quadrature(1.0 - xe, J, beta) / Phi_quadrature(xe, J, beta))
    yf, xa = orc.forward(x, om, Nd, Kd, Jd), orc.adjoint(y, om, Nd, Kd, Jd)
    e_f, e_a = rel(yf, A @ x.ravel()), rel(xa.ravel(), A.conj().T @ y)
    assert alias / 4 < e_f < 3 * alias, (sigma, J, alias, e_f)
    assert alias / 4 < e_a < 3 * alias, (sigma, J, alias, e_a)
    assert abs(np.vdot(yf, y) - np.vdot(x, xa)) / abs(np.vdot(yf, y)) < 1e-10


def test_scaling_factors_at_sigma_against_quadrature():
    for N, K, J in [(20, 32, 6), (48, 64, 4), (16, 64, 6)]:
        beta = orc.kb_beta(J, K / N)
        s = orc.scaling_factors(N, K, J)
        for n in (0, N // 2, N - 1, N // 3):
            assert s[n] == pytest.approx(1.0 / Phi_quadrature((n - N / 2.0) / K, J, beta), rel=1e-9)
