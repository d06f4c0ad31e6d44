"""GPU parity at kernel widths other than Jd = 6 (SURVEY 8(f)-4 "other Jd"): forward, adjoint and
A^H A, batches, the solvers and the "next" rows on plans with J = 2..8, element by element against the float64 oracle
on the same seeded inputs (relative L2 <= 2e-5 for the transforms, <= 1e-4 for solver output; BASELINE.json north star).
These plans run the direct V / atomic V^H kernels (interp_direct_kernel<D, J>, gridding_atomic_kernel<D, J>).
"""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import next_oracle as nxt
from oracle import nufft_oracle as orc
from oracle import solvers_oracle as sol

from parity_helpers import check_density_weights

pytestmark = pytest.mark.gpu
TOL = 2e-5
WIDTHS = [2, 3, 4, 5, 7, 8]


def rel(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.complex64)).cuda()


def host(t):
    return t.detach().cpu().numpy()


def make_plan(cfg, **kw):
    import paper_1710_03197_b200 as nb
    return nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], **kw)


def width_cfg(Nd, M, J, seed):
    rng = np.random.default_rng(seed)
    d = len(Nd)
    om = rng.uniform(-np.pi, np.pi, (M, d))
    # seam, origin, exact grid points (one weight is exactly zero, reading R6), values outside [-pi, pi) (wrapped)
    om[0] = -np.pi
    om[1] = 0.0
    om[2] = [2 * np.pi * 3 / (2 * n) for n in Nd]
    om[3] = np.pi - 1e-9
    om[4] = 7.0
    return dict(Nd=tuple(Nd), Kd=tuple(2 * n for n in Nd), Jd=(J,) * d, om=om)


def check(cfg, batch=1, **kw):
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    p = make_plan(cfg, max_batch=batch, **kw)
    x = np.stack([wl.image_gaussian(Nd, seed=wl.SEED_IMAGE + b) for b in range(batch)])
    y = np.stack([wl.data_gaussian(om.shape[0], seed=wl.SEED_Y + b) for b in range(batch)])
    yg, xg, sg = host(p.forward(dev(x))), host(p.adjoint(dev(y))), host(p.selfadjoint(dev(x)))
    errs = []
    for b in range(batch):
        yo = orc.forward(x[b].astype(np.complex128), om, Nd, Kd, Jd)
        xo = orc.adjoint(y[b].astype(np.complex128), om, Nd, Kd, Jd)
        so = orc.adjoint(yo, om, Nd, Kd, Jd)
        errs += [rel(yg[b], yo), rel(xg[b], xo), rel(sg[b], so)]
    p.destroy()
    assert max(errs) < TOL, (Jd, errs)


@pytest.mark.parametrize("J", WIDTHS)
def test_transforms_2d_at_width(J):
    check(width_cfg((64, 32), 9001, J, seed=100 + J))          # several tiles, ragged tail, non-square


@pytest.mark.parametrize("J", WIDTHS)
def test_transforms_1d_and_3d_at_width(J):
    check(width_cfg((128,), 1001, J, seed=200 + J), batch=3)
    check(width_cfg((16, 32, 16), 5003, J, seed=300 + J), batch=2)


@pytest.mark.parametrize("J", [4, 8])
def test_radial_config2_at_width(J):
    cfg = dict(wl.config(1, scale=2))                         # 128^2 golden-angle radial
    cfg["Jd"] = (J, J)
    check(cfg, batch=13)                                      # above the interleaved path's threshold: stays planar


def test_generic_kernels_at_width_6():
    """interp_mode = 2 runs the same generic kernels at J = 6: oracle parity, and agreement with the tuned kernels."""
    cfg = width_cfg((64, 64), 7000, 6, seed=5)
    check(cfg, batch=2, interp_mode=2)
    pa, pb = make_plan(cfg), make_plan(cfg, interp_mode=2)
    x = dev(wl.image_gaussian(cfg["Nd"])[None])
    assert rel(host(pb.selfadjoint(x)), host(pa.selfadjoint(x))) < 2e-6
    pa.destroy(); pb.destroy()


def test_unsupported_widths_are_refused():
    import paper_1710_03197_b200 as nb
    cfg = width_cfg((32, 32), 100, 4, seed=1)
    for Jd in [(1, 1), (9, 9), (4, 6)]:
        with pytest.raises(Exception):
            nb.NufftPlan(cfg["Nd"], cfg["Kd"], Jd, cfg["om"])
    with pytest.raises(Exception):
        make_plan(cfg, adjoint_mode=1)                        # the deterministic V^H exists for J = 6 only


@pytest.mark.parametrize("J", [4, 7])
def test_solvers_at_width(J):
    Nd = (32, 32)
    cfg = width_cfg(Nd, 4 * 32 * 32 * 2, J, seed=40 + J)
    Kd, Jd, om = cfg["Kd"], cfg["Jd"], cfg["om"]
    p = make_plan(cfg, max_batch=2)
    xt = wl.phantom(Nd)
    y = orc.forward(xt.astype(np.complex128), om, Nd, Kd, Jd)
    y = (y + wl.noise_like(y)).astype(np.complex64)
    AHA = lambda z: orc.selfadjoint(z, om, Nd, Kd, Jd)
    AHy = orc.adjoint(y.astype(np.complex128), om, Nd, Kd, Jd)
    for niter in (1, 8):
        xo, _ = sol.cg(AHA, AHy, niter)
        assert rel(host(p.solve_cg(dev(y), niter)), xo) < 1e-4
    # the paper's k-space CG (eqs. 8-11): the inverse scaling factors depend on J too
    xo, _ = nxt.cg_kspace(y.astype(np.complex128), om, Nd, Kd, Jd, 3)
    assert rel(host(p.solve_cg_kspace(dev(y), 3)), xo) < 1e-4
    # density weights (eq. 6), one iteration
    # density weights (eq. 6), one iteration: w itself against the oracle, with the bound of tests/parity_helpers.py
    # (the division by |A A^H 1| amplifies the 2e-7 operator rounding where that magnitude is small), and |A A^H 1| = 1 / w
    wo = nxt.density_weights(om, Nd, Kd, Jd, 1)
    wg = host(p.density_weights(1)).real
    check_density_weights(wg, wo, om, Nd, Kd, Jd, 1, TOL)
    assert rel(1.0 / wg, 1.0 / wo) < TOL
    p.destroy()


@pytest.mark.parametrize("J", [4, 8])
def test_toeplitz_at_width(J):
    Nd = (32, 32)
    cfg = width_cfg(Nd, 6000, J, seed=60 + J)
    Kd, Jd, om = cfg["Kd"], cfg["Jd"], cfg["om"]
    p = make_plan(cfg)
    p.toeplitz_build()
    x = wl.image_gaussian(Nd)
    That, _ = nxt.toeplitz_kernel(om, Nd, Kd, Jd)
    ref = nxt.selfadjoint_toeplitz(x.astype(np.complex128), That, Nd)
    got = host(p.selfadjoint_toeplitz(dev(x[None])))[0]
    assert rel(got, ref) < TOL
    p.destroy()
