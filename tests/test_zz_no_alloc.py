"""nufft_adjoint_noalloc (include/nufft.h): the allocation-free adjoint whose workspace grid is a file-scope `static __device__`
array of the library (2 MiB, NUFFT_NOALLOC_MAX_CELLS complex64 cells).  Checked against the existing path, nufft_adjoint
(itself compared with the float64 oracle in test_gpu_parity.py), with the criterion of every transform test: relative
L2 <= 2e-5 AND max-abs <= 50 eps32 sqrt(prod J).  Calls are made back to back because the array is shared and keeps the
previous call's contents: a large grid followed by a small one, other inputs, other plans.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

import paper_1710_03197_b200 as nb
import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 2e-5
MAX_CELLS = 262144          # NUFFT_NOALLOC_MAX_CELLS


def tol_max(Jd):
    return 50.0 * 1.1920929e-07 * float(np.sqrt(np.prod(Jd)))


def close(a, ref, Jd):
    a = a.detach().cpu().numpy().ravel().astype(np.complex128)
    ref = ref.detach().cpu().numpy().ravel().astype(np.complex128)
    e2 = np.linalg.norm(a - ref) / np.linalg.norm(ref)
    em = np.abs(a - ref).max() / np.abs(ref).max()
    assert e2 < TOL and em < tol_max(Jd), (e2, em)
    return e2, em


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.complex64)).cuda()


def plan_of(cfg, **kw):
    return nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=1, **kw)


def test_no_alloc_adjoint_matches_the_existing_adjoint_on_calls_in_a_row():
    big = wl.config(1)                      # 256^2 image, 512^2 grid = exactly MAX_CELLS, golden-angle radial, M = 131072
    small = wl.config(0)                    # 64^2 image, 128^2 grid, uniform random samples
    assert int(np.prod(big["Kd"])) == MAX_CELLS
    pb, ps = plan_of(big), plan_of(small)
    try:
        yb = [dev(wl.data_gaussian(pb.M, seed=900 + i)) for i in range(2)]
        ys = [dev(wl.data_gaussian(ps.M, seed=910 + i)) for i in range(2)]
        ref_b = [pb.adjoint(y[None])[0].clone() for y in yb]
        ref_s = [ps.adjoint(y[None])[0].clone() for y in ys]
        xb = torch.empty(big["Nd"], dtype=torch.complex64, device="cuda")
        xs = torch.empty(small["Nd"], dtype=torch.complex64, device="cuda")
        # two calls in a row on the same plan, other data: the second must not see the first one's grid
        for i in range(2):
            xb.fill_(float("nan"))
            pb.adjoint_noalloc(yb[i], xb)
            close(xb, ref_b[i], big["Jd"])
        # a small grid right after the large one (the array still holds the large grid), twice, then the large one again
        for i in range(2):
            xs.fill_(float("nan"))
            ps.adjoint_noalloc(ys[i], xs)
            close(xs, ref_s[i], small["Jd"])
        xb.fill_(float("nan"))
        pb.adjoint_noalloc(yb[0], xb)
        close(xb, ref_b[0], big["Jd"])
        # no device memory is taken by further calls (the library's cudaMalloc would show up here; torch allocates nothing)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for i in range(2):
            pb.adjoint_noalloc(yb[i], xb)
            ps.adjoint_noalloc(ys[i], xs)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= free0
        close(xb, ref_b[1], big["Jd"])
        close(xs, ref_s[1], small["Jd"])
    finally:
        pb.destroy()
        ps.destroy()


def test_no_alloc_adjoint_3d_1d_and_other_widths():
    cases = []
    c3 = wl.config(3, scale=4)              # 32^3 image, 64^3 grid = exactly MAX_CELLS, kooshball
    assert int(np.prod(c3["Kd"])) == MAX_CELLS
    cases.append(c3)
    cases.append(dict(Nd=(256,), Kd=(512,), Jd=(6,), om=wl.traj_uniform(3000, 1, seed=921)))
    cases.append(dict(Nd=(64, 128), Kd=(128, 256), Jd=(4, 4), om=wl.traj_uniform(5000, 2, seed=922)))   # generic width
    for cfg in cases:
        p = plan_of(cfg)
        try:
            x = torch.empty(cfg["Nd"], dtype=torch.complex64, device="cuda")
            for i in range(2):
                y = dev(wl.data_gaussian(p.M, seed=930 + i))
                ref = p.adjoint(y[None])[0].clone()
                x.fill_(float("nan"))
                p.adjoint_noalloc(y, x)
                close(x, ref, cfg["Jd"])
        finally:
            p.destroy()


def test_no_alloc_adjoint_refuses_what_it_cannot_serve():
    # a 1024^2 grid is beyond the static array: a clear error, nothing launched
    p = nb.NufftPlan((512, 512), (1024, 1024), (6, 6), wl.traj_uniform(2000, 2, seed=940), max_batch=1)
    try:
        x = torch.zeros((512, 512), dtype=torch.complex64, device="cuda")
        with pytest.raises(nb.NufftError) as ei:
            p.adjoint_noalloc(dev(wl.data_gaussian(p.M, seed=941)), x)
        assert ei.value.code == -6 and "NUFFT_NOALLOC_MAX_CELLS" in str(ei.value)
        torch.cuda.synchronize()
        assert float(x.abs().max()) == 0.0
    finally:
        p.destroy()
    # the deterministic mode allocates its slabs on first use: refused
    cfg = wl.config(0)
    p = plan_of(cfg, adjoint_mode=1)
    try:
        x = torch.zeros(cfg["Nd"], dtype=torch.complex64, device="cuda")
        with pytest.raises(nb.NufftError) as ei:
            p.adjoint_noalloc(dev(wl.data_gaussian(p.M, seed=942)), x)
        assert ei.value.code == -1
    finally:
        p.destroy()
