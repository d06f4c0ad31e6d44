"""GPU parity of plans with the min-max interpolator (opts.kernel = 1; "the default kernel is the
min-max kernel"; reading R25) against oracle/minmax_oracle.py, element by element on the same
seeded inputs: relative L2 <= 2e-5 for forward, adjoint and A^H A, <= 1e-4 for solver output (BASELINE.json north star).
Every kernel family is covered: planar 2-D (direct V, tiled V^H, both adjoint modes), interleaved 2-D (caller-order and
sorted V, gather-form V^H with the float64 table), 3-D tiled, 1-D, and the generic-width kernels.
"""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import minmax_oracle as mm
from oracle import nufft_oracle as orc
from oracle import solvers_oracle as sol

pytestmark = pytest.mark.gpu
TOL = 2e-5


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
    return nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], kernel="minmax", **kw)


def rand_cfg(Nd, M, J=6, seed=0):
    rng = np.random.default_rng(seed)
    d = len(Nd)
    om = rng.uniform(-np.pi, np.pi, (M, d))
    om[0] = -np.pi                      # seam
    om[1] = 0.0                         # on a grid point: delta = 0, where Kaiser-Bessel would zero a weight and min-max does not
    om[2] = [2 * np.pi * 3 / (2 * n) for n in Nd]
    om[3] = np.pi - 1e-9
    om[4] = 7.0                         # wrapped
    return dict(Nd=tuple(Nd), Kd=tuple(2 * n for n in Nd), Jd=(J,) * d, om=om)


def check(cfg, batch=1, imgs=(0,), **kw):
    Nd, Kd, Jd, om = cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"]
    p = make_plan(cfg, max_batch=batch, **kw)
    x = wl.image_gaussian(Nd, batch=batch) if batch > 1 else wl.image_gaussian(Nd)[None]
    y = wl.data_gaussian(om.shape[0], batch=batch) if batch > 1 else wl.data_gaussian(om.shape[0])[None]
    yg, xg, sg = host(p.forward(dev(x))), host(p.adjoint(dev(y))), host(p.selfadjoint(dev(x)))
    for b in imgs:
        yo = mm.forward(x[b].astype(np.complex128), om, Nd, Kd, Jd)
        xo = mm.adjoint(y[b].astype(np.complex128), om, Nd, Kd, Jd)
        so = mm.adjoint(yo, om, Nd, Kd, Jd)
        errs = (rel(yg[b], yo), rel(xg[b], xo), rel(sg[b], so))
        assert max(errs) < TOL, (b, errs)
    p.destroy()
    return x, yg


def test_minmax_planar_2d_both_adjoint_modes_and_option_acts():
    cfg = rand_cfg((64, 64), 9001, seed=1)
    x, yg = check(cfg)
    check(cfg, adjoint_mode=1)
    check(cfg, batch=3, imgs=(0, 2))
    # the option changes the operator: the Kaiser-Bessel oracle is NOT matched to the tolerance
    yk = orc.forward(x[0].astype(np.complex128), cfg["om"], cfg["Nd"], cfg["Kd"], cfg["Jd"])
    assert rel(yg[0], yk) > 2e-6


def test_minmax_interleaved_radial_and_random():
    check(dict(wl.config(1, scale=2)), batch=20, imgs=(0, 19))                      # coherent: caller-order V
    check(dict(wl.config(1, scale=2)), batch=20, imgs=(7,), interp_mode=1)          # sorted walk + layout pass
    check(rand_cfg((64, 64), 7001, seed=2), batch=40, imgs=(0, 31, 32, 39))


def test_minmax_config2_full_size_batch64_bench_configuration():
    cfg = dict(wl.config(1))
    check(cfg, batch=64, imgs=(63,))
    check(cfg)


def test_minmax_3d_tiled_direct_and_1d():
    cfg = rand_cfg((32, 32, 32), 20011, seed=3)
    check(cfg)
    check(cfg, interp_mode=1, adjoint_mode=1)
    check(dict(wl.config(3, scale=4)))                                              # kooshball 32^3
    check(rand_cfg((128,), 1001, seed=4), batch=3, imgs=(0, 2))


@pytest.mark.parametrize("J", [2, 4, 5, 8])
def test_minmax_other_widths(J):
    check(rand_cfg((32, 32), 4001, J=J, seed=10 + J))
    check(rand_cfg((16, 16, 16), 3001, J=J, seed=20 + J))


def test_minmax_non_square_images():
    """The min-max weights depend on N_a: one weight polynomial per axis."""
    check(rand_cfg((32, 64), 5001, seed=40))
    check(rand_cfg((32, 64), 5001, seed=41), batch=17, imgs=(0, 16))          # interleaved path: per-axis float64 table
    check(rand_cfg((16, 32, 64), 9001, seed=42))


def test_minmax_cg_and_toeplitz_consistency():
    Nd = (32, 32)
    cfg = rand_cfg(Nd, 4 * 32 * 32 * 2, seed=30)
    Kd, Jd, om = cfg["Kd"], cfg["Jd"], cfg["om"]
    p = make_plan(cfg)
    xt = wl.phantom(Nd)
    y = mm.forward(xt.astype(np.complex128), om, Nd, Kd, Jd)
    y = (y + wl.noise_like(y)).astype(np.complex64)
    AHA = lambda z: mm.selfadjoint(z, om, Nd, Kd, Jd)
    AHy = mm.adjoint(y.astype(np.complex128), om, Nd, Kd, Jd)
    for niter in (1, 8):
        xo, _ = sol.cg(AHA, AHy, niter)
        assert rel(host(p.solve_cg(dev(y), niter)), xo) < 1e-4
    # Toeplitz form built from this plan's own adjoint: agrees with the back-to-back operator to the kernel error
    p.toeplitz_build()
    x = wl.image_gaussian(Nd)[None]
    assert rel(host(p.selfadjoint_toeplitz(dev(x))), host(p.selfadjoint(dev(x)))) < 1e-4
    p.destroy()


def test_plan_modes_report_what_the_plan_chose():
    import paper_1710_03197_b200 as nb
    cfg = dict(wl.config(1, scale=2))                         # radial: coherent
    p = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=16)
    i = p.info()
    assert i["J"] == 6 and i["kernel"] == "kb" and i["interleaved"] and i["caller_order_interp"]
    assert not i["generic_width_kernels"] and not i["toeplitz"] and 0 < i["poly_err"] < 1e-7
    p.toeplitz_build()
    p.toeplitz_enable(True)
    assert p.info()["toeplitz"]
    p.destroy()
    cfg = rand_cfg((32, 32), 500, J=4)
    p = make_plan(cfg, max_batch=16)
    i = p.info()
    assert i["J"] == 4 and i["kernel"] == "minmax" and i["generic_width_kernels"] and not i["interleaved"]
    assert 0 < i["poly_err"] < 1e-7
    p.destroy()
