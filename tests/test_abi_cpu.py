"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU, and exports every
symbol include/nufft.h declares.  No compute calls are made here."""
import ctypes
import os
import re

import pytest

import paper_1710_03197_b200 as nb


def _declared_symbols(repo_root):
    text = open(os.path.join(repo_root, "include", "nufft.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = set(re.findall(r"\b(nufft_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_are_exported(repo_root):
    L = nb.lib()
    declared = _declared_symbols(repo_root)
    assert len(declared) >= 20
    missing = [s for s in declared if not hasattr(L, s)]
    assert missing == []
    assert sorted(nb.EXPORTED_SYMBOLS) == declared


def test_library_is_in_tree_and_is_sm100a(repo_root):
    path = nb.lib_path()
    assert os.path.commonpath([path, repo_root]) == repo_root
    assert "sm_100a" in nb.version()


def test_strerror_and_arg_validation_without_gpu():
    L = nb.lib()
    assert L.nufft_strerror(0) == b"ok"
    assert b"invalid" in L.nufft_strerror(-1)
    # argument validation happens before any CUDA call
    h = ctypes.c_void_p()
    Nd = (ctypes.c_int64 * 2)(64, 64)
    Kd = (ctypes.c_int64 * 2)(128, 128)
    Jd = (ctypes.c_int * 2)(6, 6)
    Jd_bad = (ctypes.c_int * 2)(4, 6)
    Kd_bad = (ctypes.c_int64 * 2)(96, 128)
    assert L.nufft_plan(4, Nd, Kd, Jd, 0, None, 1, None, ctypes.byref(h)) == -1          # d
    assert L.nufft_plan(2, Nd, Kd, Jd_bad, 0, None, 1, None, ctypes.byref(h)) == -1      # Jd not uniform
    for j in (1, 9):                                                                      # Jd outside 2..8
        assert L.nufft_plan(2, Nd, Kd, (ctypes.c_int * 2)(j, j), 0, None, 1, None, ctypes.byref(h)) == -1
    from paper_1710_03197_b200.binding import NufftOpts
    o = NufftOpts()
    assert L.nufft_default_opts(ctypes.byref(o)) == 0 and o.kernel == 0 and o.adjoint_mode == 0
    o.kernel = 2                                                                          # unknown interpolator
    assert L.nufft_plan(2, Nd, Kd, Jd, 0, None, 1, ctypes.byref(o), ctypes.byref(h)) == -1
    for nd in ((64, 63), (128, 64), (0, 64), (130, 64)):                                  # N odd, N >= K, N < 2
        Nd_r = (ctypes.c_int64 * 2)(*nd)
        assert L.nufft_plan(2, Nd_r, Kd, Jd, 0, None, 1, None, ctypes.byref(h)) == -1
    o.kernel, o.adjoint_mode = 0, 1                                                       # deterministic V^H is J = 6 only
    assert L.nufft_plan(2, Nd, Kd, (ctypes.c_int * 2)(4, 4), 0, None, 1, ctypes.byref(o), ctypes.byref(h)) == -1
    assert L.nufft_plan(2, Nd, Kd_bad, Jd, 0, None, 1, None, ctypes.byref(h)) == -1      # Kd != 2 Nd / not pow2
    assert L.nufft_plan(2, Nd, Kd, Jd, 0, None, 0, None, ctypes.byref(h)) == -1          # max_batch
    assert L.nufft_plan(2, Nd, Kd, Jd, 5, None, 1, None, ctypes.byref(h)) == -1          # om null with M > 0
    assert h.value is None
    assert L.nufft_forward(None, 1, None, None, None) == -1
    assert L.nufft_destroy(None) == -1
    assert L.nufft_launch_count(None) == -1


def test_binding_refuses_cpu_tensors():
    import torch
    from paper_1710_03197_b200 import binding
    with pytest.raises(TypeError):
        binding._dev(torch.zeros(4, dtype=torch.complex64), "x")
