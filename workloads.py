"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the NUFFT method's arithmetic (no kernel, no scaling factor, no FFT, no
interpolation): only images, phantoms, coil maps, noise and sample-location trajectories, generated with
numpy.random.default_rng(seed).  It imports neither oracle/ nor the CUDA package.

The shapes, sizes and structure follow BASELINE.json's five configs; they stand in
for the paper's brain template [14] and PROPELLER trajectory [15], which are not available.
Recipes are restated in DESIGN.md ("Input recipe").

om is always float64 [M][d], radians per image sample in [-pi, pi), axis a of om pairs with image axis a.
"""
import numpy as np

SEED_IMAGE, SEED_Y, SEED_OM, SEED_NOISE, SEED_COILS, SEED_PHANTOM, SEED_KOOSH = (
    1001, 1002, 1003, 1004, 1005, 1006, 1007)

GOLDEN_ANGLE = np.pi * (np.sqrt(5.0) - 1.0) / 2.0  # 111.246 degrees


# ----------------------------------------------------------------------------------------------------------
# images and data vectors
# ----------------------------------------------------------------------------------------------------------
def image_gaussian(Nd, seed=SEED_IMAGE, batch=None):
    """complex64 image(s), real and imaginary parts i.i.d. N(0,1)."""
    rng = np.random.default_rng(seed)
    shape = tuple(Nd) if batch is None else (int(batch),) + tuple(Nd)
    re = rng.standard_normal(shape)
    im = rng.standard_normal(shape)
    return (re + 1j * im).astype(np.complex64)


def data_gaussian(M, seed=SEED_Y, batch=None):
    """complex64 k-space data vector(s) y, real and imaginary parts i.i.d. N(0,1)."""
    rng = np.random.default_rng(seed)
    shape = (int(M),) if batch is None else (int(batch), int(M))
    re = rng.standard_normal(shape)
    im = rng.standard_normal(shape)
    return (re + 1j * im).astype(np.complex64)


def phantom(Nd, seed=SEED_PHANTOM, nellipses=10):
    """Shepp-Logan-like piecewise-constant 2-D phantom: sum of seeded ellipses on [-1,1]^2.  complex64 (imag=0)."""
    assert len(Nd) == 2
    rng = np.random.default_rng(seed)
    ax0 = (np.arange(Nd[0]) - Nd[0] / 2.0) / (Nd[0] / 2.0)
    ax1 = (np.arange(Nd[1]) - Nd[1] / 2.0) / (Nd[1] / 2.0)
    X0, X1 = np.meshgrid(ax0, ax1, indexing="ij")
    img = np.zeros(tuple(Nd), dtype=np.float64)
    for _ in range(nellipses):
        c = rng.uniform(-0.5, 0.5, size=2)
        semi = rng.uniform(0.05, 0.4, size=2)
        ang = rng.uniform(0.0, np.pi)
        val = rng.uniform(-0.5, 1.0)
        ca, sa = np.cos(ang), np.sin(ang)
        r0 = (X0 - c[0]) * ca + (X1 - c[1]) * sa
        r1 = -(X0 - c[0]) * sa + (X1 - c[1]) * ca
        img += val * ((r0 / semi[0]) ** 2 + (r1 / semi[1]) ** 2 <= 1.0)
    return img.astype(np.complex64)


def noise_like(y, sigma_rel=0.01, seed=SEED_NOISE):
    """Complex Gaussian noise with total std sigma_rel * rms(y) (re and im each sigma/sqrt 2). complex128."""
    rng = np.random.default_rng(seed)
    y = np.asarray(y)
    sigma = sigma_rel * np.sqrt(np.mean(np.abs(y) ** 2))
    return (sigma / np.sqrt(2.0)) * (rng.standard_normal(y.shape) + 1j * rng.standard_normal(y.shape))


def coil_maps(nc, Nd, seed=SEED_COILS):
    """Smooth Gaussian-bump complex coil sensitivities c[nc, N0, N1], sum_i |c_i|^2 = 1.  complex64.

    c_i(r) = exp(-|r - r_i|^2 / (2 s^2)) exp(i (phi_i + a_i . r)), centres on a circle of radius 0.6 N at angles
    2 pi i / nc + jitter, s = 0.35 N.
    """
    assert len(Nd) == 2
    rng = np.random.default_rng(seed)
    N0, N1 = int(Nd[0]), int(Nd[1])
    r0 = np.arange(N0) - N0 / 2.0
    r1 = np.arange(N1) - N1 / 2.0
    R0, R1 = np.meshgrid(r0, r1, indexing="ij")
    jitter = rng.uniform(-0.1, 0.1, size=nc)
    phi = rng.uniform(0.0, 2.0 * np.pi, size=nc)
    a = rng.uniform(-1.0, 1.0, size=(nc, 2)) * (np.pi / max(N0, N1))
    c = np.zeros((nc, N0, N1), dtype=np.complex128)
    for i in range(nc):
        ang = 2.0 * np.pi * i / nc + jitter[i]
        c0, c1 = 0.6 * N0 * np.cos(ang), 0.6 * N1 * np.sin(ang)
        mag = np.exp(-((R0 - c0) ** 2 / (2.0 * (0.35 * N0) ** 2) + (R1 - c1) ** 2 / (2.0 * (0.35 * N1) ** 2)))
        c[i] = mag * np.exp(1j * (phi[i] + a[i, 0] * R0 + a[i, 1] * R1))
    c /= np.sqrt(np.sum(np.abs(c) ** 2, axis=0, keepdims=True))
    return c.astype(np.complex64)


# ----------------------------------------------------------------------------------------------------------
# trajectories
# ----------------------------------------------------------------------------------------------------------
def traj_uniform(M, d, seed=SEED_OM):
    """M locations i.i.d. uniform in [-pi, pi)^d."""
    rng = np.random.default_rng(seed)
    return rng.uniform(-np.pi, np.pi, size=(int(M), int(d)))


def traj_radial_golden(nspokes, nread):
    """2-D golden-angle radial: spoke s at angle s * 111.246 deg, readout r_i = -pi + 2 pi i / nread."""
    s = np.arange(nspokes, dtype=np.float64)
    theta = s * GOLDEN_ANGLE
    r = -np.pi + 2.0 * np.pi * np.arange(nread, dtype=np.float64) / nread
    om = np.empty((nspokes, nread, 2), dtype=np.float64)
    om[:, :, 0] = r[None, :] * np.cos(theta)[:, None]
    om[:, :, 1] = r[None, :] * np.sin(theta)[:, None]
    return om.reshape(-1, 2)


def traj_spiral_vd(nleaves, npts, nturns=8.0):
    """2-D variable-density spiral: r = pi t, theta = 2 pi (nturns t + l / nleaves), t = i / npts (density ~ 1/|k|)."""
    t = np.arange(npts, dtype=np.float64) / npts
    l = np.arange(nleaves, dtype=np.float64)
    r = np.pi * t
    theta = 2.0 * np.pi * (nturns * t[None, :] + l[:, None] / nleaves)
    om = np.empty((nleaves, npts, 2), dtype=np.float64)
    om[:, :, 0] = r[None, :] * np.cos(theta)
    om[:, :, 1] = r[None, :] * np.sin(theta)
    return om.reshape(-1, 2)


def traj_propeller(nblades, nlines, nread, N):
    """2-D PROPELLER: nblades rectangular strips through the origin, blade b rotated by pi b / nblades; a blade has
    nlines parallel readouts of nread points, line spacing and readout spacing 2 pi / N (Nyquist for an N-pixel image).
    Synthetic stand-in for the non-Cartesian k-space of the paper's brain simulation (its ref. [15]),
    which is not in this container.  Sample order: blade, line, readout point."""
    dk = 2.0 * np.pi / float(N)
    kx = (np.arange(nread, dtype=np.float64) - nread / 2.0) * dk
    ky = (np.arange(nlines, dtype=np.float64) - (nlines - 1) / 2.0) * dk
    om = np.empty((nblades, nlines, nread, 2), dtype=np.float64)
    for b in range(nblades):
        th = np.pi * b / nblades
        c, s_ = np.cos(th), np.sin(th)
        om[b, :, :, 0] = c * kx[None, :] - s_ * ky[:, None]
        om[b, :, :, 1] = s_ * kx[None, :] + c * ky[:, None]
    return om.reshape(-1, 2)


def config_propeller(scale=1):
    """The paper's own experiment shape (512 x 512 image, non-Cartesian k-space of ref. [15]): Nd = 512^2,
    Kd = 1024^2, Jd = 6, PROPELLER with 24 blades x 32 lines x 512 readout points (M = 393216).  Not a BASELINE config:
    bench context leg and one parity case."""
    s = int(scale)
    N = 512 // s
    return dict(name="paper_2_3_propeller", Nd=(N, N), Kd=(2 * N, 2 * N), Jd=(6, 6),
                om=traj_propeller(max(24 // s, 3), max(32 // s, 2), N, N), ncoil=0)


def traj_kooshball(nspokes, nread, seed=SEED_KOOSH):
    """3-D radial kooshball: spokes through the origin, directions by spiral phyllotaxis on the upper hemisphere."""
    rng = np.random.default_rng(seed)
    phi0 = 2.0 * np.pi * rng.uniform()
    s = np.arange(nspokes, dtype=np.float64)
    z = (s + 0.5) / nspokes
    rho = np.sqrt(1.0 - z * z)
    az = s * np.pi * (3.0 - np.sqrt(5.0)) + phi0
    dirs = np.stack([rho * np.cos(az), rho * np.sin(az), z], axis=1)
    r = -np.pi + 2.0 * np.pi * np.arange(nread, dtype=np.float64) / nread
    om = r[None, :, None] * dirs[:, None, :]
    return om.reshape(-1, 3)


# ----------------------------------------------------------------------------------------------------------
# BASELINE.json configs (index = position in BASELINE.json "configs") and scaled-down test versions
# ----------------------------------------------------------------------------------------------------------
def config(i, scale=1):
    """Geometry + trajectory of BASELINE config i (0-based).  scale>1 divides every Nd (and spoke/readout counts)
    by `scale`, keeping the structure, for test cases the oracle finishes in seconds.

    Returns dict(name, Nd, Kd, Jd, om, ncoil).
    """
    s = int(scale)
    if i == 0:
        N = 64 // s
        return dict(name="cfg1_2d_tiny_uniform", Nd=(N, N), Kd=(2 * N, 2 * N), Jd=(6, 6),
                    om=traj_uniform(8192 // (s * s), 2), ncoil=0)
    if i == 1:
        N = 256 // s
        return dict(name="cfg2_2d_radial", Nd=(N, N), Kd=(2 * N, 2 * N), Jd=(6, 6),
                    om=traj_radial_golden(256 // s, 2 * N), ncoil=0)
    if i == 2:
        N = 512 // s
        return dict(name="cfg3_2d_vdspiral_cg", Nd=(N, N), Kd=(2 * N, 2 * N), Jd=(6, 6),
                    om=traj_spiral_vd(32, 8192 // (s * s), nturns=8.0 / s), ncoil=0)
    if i == 3:
        N = 128 // s
        return dict(name="cfg4_3d_kooshball", Nd=(N, N, N), Kd=(2 * N, 2 * N, 2 * N), Jd=(6, 6, 6),
                    om=traj_kooshball(4096 // (s * s), 4 * N), ncoil=0)
    if i == 4:
        N = 256 // s
        return dict(name="cfg5_2d_multicoil_l1tv", Nd=(N, N), Kd=(2 * N, 2 * N), Jd=(6, 6),
                    om=traj_radial_golden(128 // s, 2 * N), ncoil=32 if s == 1 else 8)
    raise ValueError("config index 0..4")
