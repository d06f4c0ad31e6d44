"""Pins for the oracle's kernel, its transform and the scaling factors (oracle/nufft_oracle.py).

Nothing here re-types the oracle's formula as the expected value: I0 comes from its power series summed in exact
rational arithmetic, Phi from quadrature of the defining integral, constants from tests/golden/kb_constants.txt.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import integrate

from oracle import nufft_oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "kb_constants.txt")


def golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            out[k] = float(v)
    return out


def i0_series(x, terms=80):
    """I0(x) = sum_k (x^2/4)^k / (k!)^2, exact rationals then one rounding."""
    q = Fraction(x) ** 2 / 4
    s, term = Fraction(0), Fraction(1)
    for k in range(terms):
        s += term
        term = term * q / ((k + 1) ** 2)
    return float(s)


def test_beta_and_golden_constants():
    g = golden()
    beta = orc.kb_beta(6, 2.0)
    assert beta == pytest.approx(g["beta"], rel=1e-12)
    assert i0_series(beta) == pytest.approx(g["I0_beta"], rel=1e-9)
    assert float(orc.kb_phi(1.0, 6, beta)) == pytest.approx(g["phi_1"], rel=1e-11)
    assert float(orc.kb_phi(2.0, 6, beta)) == pytest.approx(g["phi_2"], rel=1e-11)
    assert float(orc.kb_phi(2.5, 6, beta)) == pytest.approx(g["phi_2p5"], rel=1e-9)
    assert float(orc.kb_Phi(0.0, 6, beta)) == pytest.approx(g["Phi_0"], rel=1e-11)
    s = orc.scaling_factors(64, 128, 6)
    assert s[32] == pytest.approx(g["s_centre"], rel=1e-11)
    assert s[0] == pytest.approx(g["s_edge"], rel=1e-11)
    ratio = float(orc.kb_Phi(0.75, 6, beta) / orc.kb_Phi(0.25, 6, beta))
    assert abs(ratio) == pytest.approx(g["alias_edge"], rel=0.05)


@pytest.mark.parametrize("t", [0.0, 0.3, 1.0, 1.7, 2.0, 2.5, 2.99, -0.4, -2.2])
def test_phi_against_power_series(t):
    beta = orc.kb_beta(6, 2.0)
    expect = i0_series(beta * math.sqrt(1.0 - (2.0 * t / 6.0) ** 2)) / i0_series(beta)
    assert float(orc.kb_phi(t, 6, beta)) == pytest.approx(expect, rel=1e-12)


def test_phi_support_symmetry_monotone():
    beta = orc.kb_beta(6, 2.0)
    assert float(orc.kb_phi(0.0, 6, beta)) == 1.0
    for t in (3.0, -3.0, 3.5, -7.0):          # open support (reading R6)
        assert float(orc.kb_phi(t, 6, beta)) == 0.0
    t = np.linspace(0.0, 2.999, 500)
    v = orc.kb_phi(t, 6, beta)
    assert np.all(np.diff(v) < 0.0)
    assert np.array_equal(orc.kb_phi(-t, 6, beta), v)


@pytest.mark.parametrize("xi", [0.0, 0.05, 0.125, 0.25, 0.4, 0.75, 1.3])
def test_Phi_is_the_fourier_transform_of_phi(xi):
    """Phi(xi) = int_{-J/2}^{J/2} phi(t) cos(2 pi xi t) dt  by adaptive quadrature (covers both sinh and sin branches)."""
    J = 6
    beta = orc.kb_beta(J, 2.0)
    val, err = integrate.quad(lambda t: float(orc.kb_phi(t, J, beta)) * math.cos(2 * math.pi * xi * t),
                              -J / 2, J / 2, epsabs=1e-14, epsrel=1e-13, limit=400)
    assert float(orc.kb_Phi(xi, J, beta)) == pytest.approx(val, abs=5e-12)


@pytest.mark.parametrize("J,sigma", [(4, 2.0), (6, 1.5), (8, 2.0)])
def test_Phi_other_widths(J, sigma):
    beta = orc.kb_beta(J, sigma)
    for xi in (0.0, 0.5 / sigma):
        val, _ = integrate.quad(lambda t: float(orc.kb_phi(t, J, beta)) * math.cos(2 * math.pi * xi * t),
                                -J / 2, J / 2, epsabs=1e-14, epsrel=1e-13, limit=400)
        assert float(orc.kb_Phi(xi, J, beta)) == pytest.approx(val, abs=5e-12)


def test_scaling_factors_real_positive_symmetric():
    s = orc.scaling_factors(64, 128, 6)
    assert s.dtype == np.float64 and s.shape == (64,)
    assert np.all(s > 0)
    assert np.allclose(s[1:], s[1:][::-1], rtol=1e-13)      # s[n] depends on |n - N/2|
    assert np.argmin(s) == 32


def test_partition_of_unity():
    """s(0) * sum_k phi(f - k) ~ 1 for every offset f: within 1e-5 of 1; at f = 0 the two end points t = +-3 drop
    out (open support, reading R6) which gives the minimum 0.99999108 quoted in SURVEY.md section 8(c)."""
    beta = orc.kb_beta(6, 2.0)
    s0 = orc.scaling_factors(64, 128, 6)[32]
    f = np.linspace(0.0, 1.0, 1001)[:, None]
    k = np.arange(-4, 5)[None, :]
    tot = s0 * orc.kb_phi(f - k, 6, beta).sum(axis=1)
    assert np.max(np.abs(tot - 1.0)) < 1e-5
    assert tot[0] == pytest.approx(0.99999108, abs=2e-8)
    assert tot[0] == tot.min()
