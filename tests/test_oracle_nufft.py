"""Pins for the float64 NUFFT oracle (oracle/nufft_oracle.py) against what the mathematics fixes.

  * the plain definition (brute-force non-uniform DFT written out with explicit loops / dense matrices here,
    not the oracle's own ndft_* helpers, which are themselves pinned against those loops);
  * the adjoint identity; unit impulses (closed form); Cartesian samples vs numpy.fft; dense V matrix on tiny
    sizes; Hermitian / PSD structure of A^H A; Toeplitz PSF; batch and coil sums.
Chosen so that a dropped term, a wrong sign, a transposed axis or a mis-centred index fails at least one.
"""
import numpy as np
import pytest

import workloads as wl
from oracle import nufft_oracle as orc


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


def ndft_matrix(om, Nd):
    """Dense M x prod(N) matrix of the plain definition: exp(-i sum_a om[m,a] (n_a - N_a/2)), C-order columns."""
    M, d = om.shape
    cols = np.stack(np.meshgrid(*[np.arange(N) - N / 2.0 for N in Nd], indexing="ij"), axis=-1).reshape(-1, d)
    return np.exp(-1j * (om @ cols.T))


# ---------------------------------------------------------------------------------------------------------
# the brute-force helpers themselves
# ---------------------------------------------------------------------------------------------------------
def test_ndft_helpers_match_explicit_loops():
    rng = np.random.default_rng(5)
    Nd = (4, 6)
    om = rng.uniform(-np.pi, np.pi, (7, 2))
    x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
    y = rng.standard_normal(7) + 1j * rng.standard_normal(7)
    fwd = np.zeros(7, complex)
    adj = np.zeros(Nd, complex)
    for m in range(7):
        for n0 in range(4):
            for n1 in range(6):
                ph = om[m, 0] * (n0 - 2) + om[m, 1] * (n1 - 3)
                fwd[m] += x[n0, n1] * np.exp(-1j * ph)
                adj[n0, n1] += y[m] * np.exp(+1j * ph)
    assert rel(orc.ndft_forward(x, om, Nd), fwd) < 1e-14
    assert rel(orc.ndft_adjoint(y, om, Nd), adj) < 1e-14
    A = ndft_matrix(om, Nd)
    assert rel(A @ x.ravel(), fwd) < 1e-14
    Nd3 = (2, 3, 4)
    om3 = rng.uniform(-np.pi, np.pi, (5, 3))
    x3 = rng.standard_normal(Nd3) + 1j * rng.standard_normal(Nd3)
    y3 = rng.standard_normal(5) + 1j * rng.standard_normal(5)
    A3 = ndft_matrix(om3, Nd3)
    assert rel(orc.ndft_forward(x3, om3, Nd3), A3 @ x3.ravel()) < 1e-14
    assert rel(orc.ndft_adjoint(y3, om3, Nd3), (A3.conj().T @ y3).reshape(Nd3)) < 1e-14


# ---------------------------------------------------------------------------------------------------------
# forward / adjoint against the plain definition  (north star: rel L2 <= 1e-4 for Jd = 6, Kd = 2 Nd)
# ---------------------------------------------------------------------------------------------------------
def test_forward_adjoint_vs_ndft_config1():
    cfg = wl.config(0)
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    x = wl.image_gaussian(Nd).astype(np.complex128)
    y = wl.data_gaussian(om.shape[0]).astype(np.complex128)
    e_f = rel(orc.forward(x, om, Nd, Kd, Jd), orc.ndft_forward(x, om, Nd))
    e_a = rel(orc.adjoint(y, om, Nd, Kd, Jd), orc.ndft_adjoint(y, om, Nd))
    assert e_f < 1e-4 and e_a < 1e-4
    assert e_f < 2e-5 and e_a < 2e-5        # SURVEY 8(c) measured 6.6e-6; a dropped term would be >> this


def test_forward_adjoint_vs_ndft_3d_and_nonsquare():
    rng = np.random.default_rng(11)
    for Nd in [(16, 16, 16), (12, 20), (8, 10, 6)]:
        Kd = tuple(2 * n for n in Nd)
        Jd = (6,) * len(Nd)
        om = rng.uniform(-np.pi, np.pi, (300, len(Nd)))
        x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
        y = rng.standard_normal(300) + 1j * rng.standard_normal(300)
        A = ndft_matrix(om, Nd)
        assert rel(orc.forward(x, om, Nd, Kd, Jd), A @ x.ravel()) < 3e-5
        assert rel(orc.adjoint(y, om, Nd, Kd, Jd).ravel(), A.conj().T @ y) < 3e-5


def test_samples_on_boundaries_and_wrapping():
    """om exactly at -pi, 0, on grid points, and outside [-pi,pi) (wrapped by periodicity of the grid)."""
    Nd, Kd, Jd = (16, 12), (32, 24), (6, 6)
    om = np.array([[-np.pi, -np.pi], [0.0, 0.0], [np.pi - 1e-9, 0.3], [2 * np.pi / 32 * 5, -2 * np.pi / 24 * 3],
                   [-np.pi, 1.0], [3.0, -3.1]])
    rng = np.random.default_rng(2)
    x = rng.standard_normal(Nd) + 1j * rng.standard_normal(Nd)
    A = ndft_matrix(om, Nd)
    assert rel(orc.forward(x, om, Nd, Kd, Jd), A @ x.ravel()) < 3e-5
    shifted = om + 2 * np.pi * np.array([[1, 0], [0, -1], [-1, 1], [2, 0], [0, 0], [1, 1]])
    # n - N/2 is an integer, so the exact transform is 2 pi periodic in om; the oracle must be too
    assert rel(orc.forward(x, shifted, Nd, Kd, Jd), orc.forward(x, om, Nd, Kd, Jd)) < 1e-12


def test_adjoint_identity():
    """<A x, y> = <x, A^H y> to 1e-10 (north star); fails for a normalised ifft (reading R5) or complex weights."""
    for i, scale in [(0, 1), (3, 8)]:
        cfg = wl.config(i, scale)
        Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
        x = wl.image_gaussian(Nd, seed=7).astype(np.complex128)
        y = wl.data_gaussian(om.shape[0], seed=8).astype(np.complex128)
        lhs = np.vdot(orc.forward(x, om, Nd, Kd, Jd), y)
        rhs = np.vdot(x, orc.adjoint(y, om, Nd, Kd, Jd))
        assert abs(lhs - rhs) / abs(lhs) < 1e-10


def test_unit_impulse_sign_and_centring():
    """Impulse at index N/2 -> ~1 for every om; impulse at n0 -> exp(-i om . (n0 - N/2)) (reading R4)."""
    Nd, Kd, Jd = (32, 24), (64, 48), (6, 6)
    om = wl.traj_uniform(500, 2, seed=3)
    x = np.zeros(Nd, complex)
    x[16, 12] = 1.0
    y = orc.forward(x, om, Nd, Kd, Jd)
    assert np.max(np.abs(y - 1.0)) < 2e-5
    for n0 in [(0, 0), (31, 23), (5, 20), (17, 12)]:
        x = np.zeros(Nd, complex)
        x[n0] = 1.0
        expect = np.exp(-1j * (om[:, 0] * (n0[0] - 16) + om[:, 1] * (n0[1] - 12)))
        assert np.max(np.abs(orc.forward(x, om, Nd, Kd, Jd) - expect)) < 3e-5


def test_cartesian_samples_reduce_to_fft():
    """om on the N-point grid 2 pi (k - N/2)/N -> fftshift(fftn(ifftshift(x))) (library routine), within the kernel
    error (KB is not an interpolating kernel; SURVEY 8(c) measured 1.3e-5)."""
    Nd, Kd, Jd = (32, 16), (64, 32), (6, 6)
    k0, k1 = np.meshgrid(np.arange(32), np.arange(16), indexing="ij")
    om = np.stack([2 * np.pi * (k0.ravel() - 16) / 32, 2 * np.pi * (k1.ravel() - 8) / 16], axis=1)
    x = wl.image_gaussian(Nd, seed=4).astype(np.complex128)
    expect = np.fft.fftshift(np.fft.fftn(np.fft.ifftshift(x)))
    assert rel(orc.forward(x, om, Nd, Kd, Jd).reshape(Nd), expect) < 1e-4
    y = wl.data_gaussian(om.shape[0], seed=5).astype(np.complex128).reshape(Nd)
    expect_adj = np.fft.fftshift(np.fft.ifftn(np.fft.ifftshift(y))) * y.size
    assert rel(orc.adjoint(y.ravel(), om, Nd, Kd, Jd), expect_adj) < 1e-4


# ---------------------------------------------------------------------------------------------------------
# stages
# ---------------------------------------------------------------------------------------------------------
def test_fft_stage_against_dft_matrix():
    """scale_pad_fft = (DFT matrix of size K) applied per axis to the circularly placed s*x; O(K^2) matrices."""
    Nd, Kd, Jd = (8, 16), (16, 32), (6, 6)
    x = wl.image_gaussian(Nd, seed=9).astype(np.complex128)
    s0 = orc.scaling_factors(8, 16, 6)
    s1 = orc.scaling_factors(16, 32, 6)
    g = np.zeros(Kd, complex)
    for n0 in range(8):
        for n1 in range(16):
            g[(n0 - 4) % 16, (n1 - 8) % 32] = s0[n0] * s1[n1] * x[n0, n1]
    F0 = np.exp(-2j * np.pi * np.outer(np.arange(16), np.arange(16)) / 16)
    F1 = np.exp(-2j * np.pi * np.outer(np.arange(32), np.arange(32)) / 32)
    G = F0 @ g @ F1.T
    assert rel(orc.scale_pad_fft(x, Nd, Kd, Jd), G) < 1e-13
    # F^H, crop, S^H: conjugate-transposed matrices, no 1/prod(K)
    Gin = wl.image_gaussian(Kd, seed=10).astype(np.complex128)
    gi = F0.conj().T @ Gin @ F1.conj()
    out = np.zeros(Nd, complex)
    for n0 in range(8):
        for n1 in range(16):
            out[n0, n1] = s0[n0] * s1[n1] * gi[(n0 - 4) % 16, (n1 - 8) % 32]
    assert rel(orc.ifft_crop_scale(Gin, Nd, Kd, Jd), out) < 1e-13


def dense_V(om, Nd, Kd, Jd):
    """Dense M x prod(K) interpolation matrix built entry by entry from the reading R6 rule, with explicit loops."""
    M, d = om.shape
    V = np.zeros((M, int(np.prod(Kd))))
    for m in range(M):
        per_axis = []
        for a in range(d):
            K, J, N = Kd[a], Jd[a], Nd[a]
            beta = orc.kb_beta(J, K / N)
            u = om[m, a] * K / (2 * np.pi)
            k0 = int(np.ceil(u - J / 2))
            per_axis.append([((k0 + j) % K, float(orc.kb_phi(u - (k0 + j), J, beta))) for j in range(J)])
        if d == 2:
            for i0, w0 in per_axis[0]:
                for i1, w1 in per_axis[1]:
                    V[m, i0 * Kd[1] + i1] += w0 * w1
        else:
            for i0, w0 in per_axis[0]:
                for i1, w1 in per_axis[1]:
                    for i2, w2 in per_axis[2]:
                        V[m, (i0 * Kd[1] + i1) * Kd[2] + i2] += w0 * w1 * w2
    return V


@pytest.mark.parametrize("Nd", [(8, 6), (4, 6, 4)])
def test_interp_and_gridding_against_dense_matrix(Nd):
    Kd = tuple(2 * n for n in Nd)
    Jd = (6,) * len(Nd)
    rng = np.random.default_rng(21)
    om = rng.uniform(-np.pi, np.pi, (40, len(Nd)))
    om[0] = -np.pi                   # wraps
    om[1] = 0.0                      # exactly on a grid point: 5 active points per axis
    V = dense_V(om, Nd, Kd, Jd)
    G = rng.standard_normal(Kd) + 1j * rng.standard_normal(Kd)
    y = rng.standard_normal(40) + 1j * rng.standard_normal(40)
    assert rel(orc.interp(G, om, Nd, Kd, Jd), V @ G.ravel()) < 1e-14
    assert rel(orc.grid_adjoint(y, om, Nd, Kd, Jd).ravel(), V.T @ y) < 1e-14
    assert np.count_nonzero(V[1]) == 5 ** len(Nd)
    # each row has at most prod(J) non-zeros, all positive
    assert np.all((V > 0).sum(axis=1) <= 6 ** len(Nd)) and np.all(V >= 0)


def test_stencil_indices_and_weights():
    idx, w = orc.stencil(np.array([0.0, -np.pi, 0.1234]), 16, 32, 6)
    assert idx.shape == (3, 6) and w.shape == (3, 6)
    assert list(idx[0]) == [29, 30, 31, 0, 1, 2]          # u = 0: k0 = -3
    assert w[0, 0] == 0.0 and w[0, 3] == 1.0              # phi(3) = 0 (open support), phi(0) = 1
    assert list(idx[1]) == [13, 14, 15, 16, 17, 18]       # u = -16: k0 = -19 -> 13
    u = 0.1234 * 32 / (2 * np.pi)
    assert idx[2, 0] == int(np.ceil(u - 3)) % 32
    assert np.all(w[2] > 0)


# ---------------------------------------------------------------------------------------------------------
# A^H A, batch, coils
# ---------------------------------------------------------------------------------------------------------
def test_selfadjoint_hermitian_psd_and_composition():
    cfg = wl.config(1, 8)
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    x = wl.image_gaussian(Nd, seed=31).astype(np.complex128)
    z = wl.image_gaussian(Nd, seed=32).astype(np.complex128)
    Tx = orc.selfadjoint(x, om, Nd, Kd, Jd)
    Tz = orc.selfadjoint(z, om, Nd, Kd, Jd)
    assert np.array_equal(Tx, orc.adjoint(orc.forward(x, om, Nd, Kd, Jd), om, Nd, Kd, Jd))
    assert abs(np.vdot(x, Tz) - np.conj(np.vdot(z, Tx))) / abs(np.vdot(x, Tz)) < 1e-10
    q = np.vdot(x, Tx)
    assert abs(q.imag) / abs(q) < 1e-10 and q.real > 0
    assert q.real == pytest.approx(np.linalg.norm(orc.forward(x, om, Nd, Kd, Jd)) ** 2, rel=1e-10)


def test_selfadjoint_psf_is_toeplitz():
    """Exact operator: (A^H A x)[n] = sum_n' T[n - n'] x[n'],  T[l] = sum_m exp(i om_m . l)."""
    Nd, Kd, Jd = (8, 8), (16, 16), (6, 6)
    om = wl.traj_uniform(200, 2, seed=33)
    x = wl.image_gaussian(Nd, seed=34).astype(np.complex128)
    out = np.zeros(Nd, complex)
    for n0 in range(8):
        for n1 in range(8):
            for m0 in range(8):
                for m1 in range(8):
                    T = np.sum(np.exp(1j * (om[:, 0] * (n0 - m0) + om[:, 1] * (n1 - m1))))
                    out[n0, n1] += T * x[m0, m1]
    assert rel(orc.selfadjoint(x, om, Nd, Kd, Jd), out) < 5e-5


def test_linearity_and_coils():
    cfg = wl.config(4, 8)
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    c = wl.coil_maps(4, Nd).astype(np.complex128)
    assert np.allclose(np.sum(np.abs(c) ** 2, axis=0), 1.0, atol=1e-6)
    x = wl.image_gaussian(Nd, seed=41).astype(np.complex128)
    z = wl.image_gaussian(Nd, seed=42).astype(np.complex128)
    a = 0.3 - 1.1j
    assert rel(orc.forward(x + a * z, om, Nd, Kd, Jd),
               orc.forward(x, om, Nd, Kd, Jd) + a * orc.forward(z, om, Nd, Kd, Jd)) < 1e-13
    yc = orc.forward_coils(x, c, om, Nd, Kd, Jd)
    assert yc.shape == (4, om.shape[0])
    for i in range(4):
        assert np.array_equal(yc[i], orc.forward(c[i] * x, om, Nd, Kd, Jd))
    acc = sum(np.conj(c[i]) * orc.adjoint(yc[i], om, Nd, Kd, Jd) for i in range(4))
    assert rel(orc.adjoint_coils(yc, c, om, Nd, Kd, Jd), acc) < 1e-14
    assert rel(orc.selfadjoint_coils(x, c, om, Nd, Kd, Jd), acc) < 1e-14
    # multi-coil adjoint identity
    yr = np.stack([wl.data_gaussian(om.shape[0], seed=50 + i) for i in range(4)]).astype(np.complex128)
    lhs = np.vdot(yc, yr)
    rhs = np.vdot(x, orc.adjoint_coils(yr, c, om, Nd, Kd, Jd))
    assert abs(lhs - rhs) / abs(lhs) < 1e-10


def test_workload_generators_shapes_and_ranges():
    for i, M in [(0, 8192), (1, 131072), (2, 262144), (4, 65536)]:
        cfg = wl.config(i)
        assert cfg["om"].shape == (M, 2) and cfg["om"].dtype == np.float64
        assert cfg["om"].min() >= -np.pi - 1e-12 and cfg["om"].max() < np.pi
    cfg = wl.config(3, 4)
    assert cfg["om"].shape == (4096 // 16 * 128, 3)
    assert np.all(np.linalg.norm(cfg["om"], axis=1) <= np.pi + 1e-9)
    assert wl.config(0)["om"][0].tolist() == wl.config(0)["om"][0].tolist()      # seeded
    ph = wl.phantom((64, 64))
    assert ph.dtype == np.complex64 and len(np.unique(ph.real)) < 200
    # PROPELLER stand-in for the paper's own experiment: blades are rotated copies of a Cartesian strip
    cfg = wl.config_propeller()
    assert cfg["Nd"] == (512, 512) and cfg["om"].shape == (24 * 32 * 512, 2)
    om = cfg["om"].reshape(24, 32, 512, 2)
    dk = 2 * np.pi / 512
    assert np.allclose(np.diff(om[0, :, :, 0], axis=1), dk) and np.allclose(np.diff(om[0, :, :, 1], axis=0), dk)
    r0 = np.linalg.norm(om[0], axis=-1)
    for b in (1, 7, 23):
        assert np.allclose(np.linalg.norm(om[b], axis=-1), r0)                   # rotation keeps the radius
        ang = np.arctan2(om[b, 16, 300, 1], om[b, 16, 300, 0]) - np.arctan2(om[0, 16, 300, 1], om[0, 16, 300, 0])
        assert np.isclose((ang - np.pi * b / 24 + np.pi) % (2 * np.pi) - np.pi, 0.0, atol=1e-9)
