"""Pins for the oracle at kernel widths other than Jd = 6 (SURVEY 8(f)-4 "other Jd"; the
interpolator size J is a parameter of the method).

What fixes the expected values: the plain definition (dense non-uniform DFT matrix built here), the power series of I0
in exact rationals, and the aliasing ratio |Phi(3/4)| / Phi(1/4) obtained by QUADRATURE of the defining integral of the
kernel transform (not the oracle's closed form).  The error of the method at the image edge is that ratio (SURVEY 8(c),
"Why this derivation is right"), so the measured error must sit within a small factor of it ON BOTH SIDES for every J:
a wrong beta, a stencil shifted by one cell or a kernel evaluated at the wrong offset breaks the upper bound, and an
oracle that silently ignored J (always using 6 points) breaks the lower one.
"""
import math
from fractions import Fraction

import numpy as np
import pytest
from scipy import integrate

from oracle import nufft_oracle as orc

WIDTHS = [2, 3, 4, 5, 6, 7, 8]


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def ndft_matrix(om, Nd):
    M, d = om.shape
    cols = np.stack(np.meshgrid(*[np.arange(N) - N / 2.0 for N in Nd], indexing="ij"), axis=-1).reshape(-1, d)
    return np.exp(-1j * (om @ cols.T))


def i0_series(x, terms=90):
    q = Fraction(x) ** 2 / 4
    s, term = Fraction(0), Fraction(1)
    for k in range(terms):
        s += term
        term = term * q / ((k + 1) ** 2)
    return float(s)


def i0_float(x):
    """The same power series summed in floats (all terms positive: no cancellation), for the bulk checks."""
    q, s, term, k = 0.25 * x * x, 0.0, 1.0, 0
    while term > 1e-18 * s:
        s += term
        k += 1
        term *= q / (k * k)
    return s


def Phi_quadrature(xi, J, beta):
    """Phi(xi) = integral over (-J/2, J/2) of phi(t) cos(2 pi xi t) dt, phi from the I0 power series."""
    i0b = i0_float(beta)
    f = lambda t: i0_float(beta * math.sqrt(max(0.0, 1.0 - (2.0 * t / J) ** 2))) / i0b
    val, _ = integrate.quad(lambda t: f(t) * math.cos(2 * math.pi * xi * t), -J / 2.0, J / 2.0, limit=200,
                            epsabs=1e-13, epsrel=1e-12)
    return val


@pytest.mark.parametrize("J", WIDTHS)
def test_kernel_and_transform_at_width(J):
    beta = orc.kb_beta(J, 2.0)
    # beta = pi sqrt((J/2)^2 (3/2)^2 - 0.8) at sigma = 2 (reading R2)
    assert beta == pytest.approx(math.pi * math.sqrt(J * J * 9.0 / 16.0 - 0.8), rel=1e-14)
    for t in [0.0, 0.37 * J / 2, -0.81 * J / 2, 0.999 * J / 2]:
        expect = i0_series(beta * math.sqrt(1.0 - (2.0 * t / J) ** 2)) / i0_series(beta)
        assert float(orc.kb_phi(t, J, beta)) == pytest.approx(expect, rel=1e-11)
    assert float(orc.kb_phi(J / 2.0, J, beta)) == 0.0 and float(orc.kb_phi(-J / 2.0 - 0.1, J, beta)) == 0.0
    for xi in [0.0, 0.11, 0.25]:
        assert float(orc.kb_Phi(xi, J, beta)) == pytest.approx(Phi_quadrature(xi, J, beta), rel=1e-9)


@pytest.mark.parametrize("J", WIDTHS)
def test_stencil_covers_support_at_width(J):
    """k0 = ceil(u - J/2): the J points k0..k0+J-1 are exactly the grid points with |u - k| < J/2 (reading R6)."""
    N, K = 16, 32
    rng = np.random.default_rng(J)
    om = rng.uniform(-np.pi, np.pi, 200)
    idx, w = orc.stencil(om, N, K, J)
    u = om * K / (2 * np.pi)
    beta = orc.kb_beta(J, 2.0)
    for m in range(200):
        inside = [k for k in range(-3 * K, 3 * K) if abs(u[m] - k) < J / 2.0]
        assert len(inside) == J
        assert [k % K for k in inside] == list(idx[m])
        for j, k in enumerate(inside):
            expect = i0_float(beta * math.sqrt(1.0 - (2.0 * (u[m] - k) / J) ** 2)) / i0_float(beta)
            assert w[m, j] == pytest.approx(expect, rel=1e-10)


@pytest.mark.parametrize("J", WIDTHS)
def test_forward_adjoint_vs_ndft_at_width(J):
    rng = np.random.default_rng(11)
    Nd, Kd, Jd = (12, 20), (24, 40), (J, J)
    om = rng.uniform(-np.pi, np.pi, (300, 2))
    x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
    y = rng.standard_normal(300) + 1j * rng.standard_normal(300)
    A = ndft_matrix(om, Nd)
    beta = orc.kb_beta(J, 2.0)
    alias = abs(Phi_quadrature(0.75, J, beta) / Phi_quadrature(0.25, J, beta))
    yf = orc.forward(x, om, Nd, Kd, Jd)
    xa = orc.adjoint(y, om, Nd, Kd, Jd)
    e_f = rel(yf, A @ x.ravel())
    e_a = rel(xa.ravel(), A.conj().T @ y)
    assert alias / 4 < e_f < 3 * alias, (J, alias, e_f)
    assert alias / 4 < e_a < 3 * alias, (J, alias, e_a)
    assert abs(np.vdot(yf, y) - np.vdot(x, xa)) / abs(np.vdot(yf, y)) < 1e-10


def test_error_falls_by_about_a_decade_per_cell_of_width():
    rng = np.random.default_rng(5)
    N, K = 32, 64
    om = rng.uniform(-np.pi, np.pi, (200, 1))
    x = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    A = ndft_matrix(om, (N,))
    errs = [rel(orc.forward(x, om, (N,), (K,), (J,)), A @ x) for J in WIDTHS]
    for a, b in zip(errs, errs[1:]):
        assert 4.0 < a / b < 25.0, errs
