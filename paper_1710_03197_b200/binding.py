"""ctypes binding of include/nufft.h.  Same names as the C ABI; marshalling only (pointers, sizes, stream).

torch is used for device memory and streams; every step of the path runs in the library's CUDA kernels.
"""
import ctypes
import os

import numpy as np

from . import build as _build

_c = ctypes
_PLAN = _c.c_void_p
_PTR = _c.c_void_p
_I64P = _c.POINTER(_c.c_int64)

EXPORTED_SYMBOLS = [
    "nufft_default_opts", "nufft_plan", "nufft_forward", "nufft_adjoint", "nufft_selfadjoint", "nufft_adjoint_noalloc",
    "nufft_forward_host", "nufft_adjoint_host", "nufft_selfadjoint_host", "nufft_host_input_ready",
    "nufft_density_weights", "nufft_adjoint_dcf", "nufft_toeplitz_build", "nufft_toeplitz_enable",
    "nufft_selfadjoint_toeplitz", "nufft_selfadjoint_toeplitz_coils", "nufft_solve_l1tv_lad", "nufft_solve_cg_kspace",
    "nufft_stage_scale_fft", "nufft_stage_interp", "nufft_stage_gridding", "nufft_stage_fft_scale",
    "nufft_set_coils", "nufft_forward_coils", "nufft_adjoint_coils", "nufft_selfadjoint_coils",
    "nufft_solve_cg", "nufft_solve_l1tv_ols", "nufft_plan_info", "nufft_plan_modes", "nufft_plan_tile_histogram", "nufft_launch_count", "nufft_destroy",
    "nufft_profile_enable", "nufft_profile_reset", "nufft_profile_count", "nufft_profile_get",
    "nufft_strerror", "nufft_last_cuda_error", "nufft_version",
]


class NufftOpts(_c.Structure):
    _fields_ = [("coef_mode", _c.c_int), ("adjoint_mode", _c.c_int), ("interp_mode", _c.c_int),
                ("tile", _c.c_int * 3), ("max_subtile", _c.c_int), ("use_graphs", _c.c_int),
                ("batch_layout", _c.c_int), ("kernel", _c.c_int)]


class NufftError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__("%s failed: %d (%s)" % (what, code, _strerror(code)))


_lib = None


def lib_path():
    return _build.LIB_PATH


def lib():
    """Load (building first if needed) the C-ABI shared library.  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB_PATH
    if not os.path.exists(path) or _build.stale():
        path = _build.build()
    L = _c.CDLL(path)
    L.nufft_default_opts.argtypes = [_c.POINTER(NufftOpts)]
    L.nufft_plan.argtypes = [_c.c_int, _I64P, _I64P, _c.POINTER(_c.c_int), _c.c_int64, _c.POINTER(_c.c_double),
                             _c.c_int, _c.POINTER(NufftOpts), _c.POINTER(_PLAN)]
    for name in ("nufft_forward", "nufft_adjoint", "nufft_selfadjoint", "nufft_forward_host", "nufft_adjoint_host",
                 "nufft_selfadjoint_host", "nufft_stage_scale_fft",
                 "nufft_stage_interp", "nufft_stage_gridding", "nufft_stage_fft_scale"):
        getattr(L, name).argtypes = [_PLAN, _c.c_int, _PTR, _PTR, _PTR]
    L.nufft_adjoint_noalloc.argtypes = [_PLAN, _PTR, _PTR, _PTR]
    L.nufft_host_input_ready.argtypes = [_PLAN, _c.c_int]
    L.nufft_density_weights.argtypes = [_PLAN, _c.c_int, _PTR, _PTR]
    L.nufft_adjoint_dcf.argtypes = [_PLAN, _c.c_int, _PTR, _PTR, _PTR, _PTR]
    L.nufft_toeplitz_build.argtypes = [_PLAN, _PTR, _PTR]
    L.nufft_toeplitz_enable.argtypes = [_PLAN, _c.c_int]
    L.nufft_selfadjoint_toeplitz.argtypes = [_PLAN, _c.c_int, _PTR, _PTR, _PTR]
    L.nufft_selfadjoint_toeplitz_coils.argtypes = [_PLAN, _PTR, _PTR, _PTR]
    L.nufft_set_coils.argtypes = [_PLAN, _c.c_int, _PTR]
    for name in ("nufft_forward_coils", "nufft_adjoint_coils", "nufft_selfadjoint_coils"):
        getattr(L, name).argtypes = [_PLAN, _PTR, _PTR, _PTR]
    L.nufft_solve_cg.argtypes = [_PLAN, _c.c_int, _PTR, _PTR, _c.c_int, _c.POINTER(_c.c_double), _PTR]
    L.nufft_solve_l1tv_ols.argtypes = [_PLAN, _c.c_int, _PTR, _PTR, _c.c_double, _c.c_double, _c.c_int, _c.c_int,
                                       _c.c_int, _PTR]
    L.nufft_solve_l1tv_lad.argtypes = L.nufft_solve_l1tv_ols.argtypes
    L.nufft_solve_cg_kspace.argtypes = [_PLAN, _PTR, _PTR, _c.c_int, _c.POINTER(_c.c_double), _PTR]
    L.nufft_plan_info.argtypes = [_PLAN, _I64P, _I64P, _I64P, _I64P, _I64P]
    L.nufft_plan_modes.argtypes = [_PLAN, _c.POINTER(_c.c_int), _c.POINTER(_c.c_int), _c.POINTER(_c.c_int),
                                   _c.POINTER(_c.c_double)]
    L.nufft_plan_tile_histogram.argtypes = [_PLAN, _I64P]
    L.nufft_launch_count.argtypes = [_PLAN]
    L.nufft_launch_count.restype = _c.c_int64
    L.nufft_destroy.argtypes = [_PLAN]
    L.nufft_profile_enable.argtypes = [_PLAN, _c.c_int]
    L.nufft_profile_reset.argtypes = [_PLAN]
    L.nufft_profile_count.argtypes = [_PLAN]
    L.nufft_profile_get.argtypes = [_PLAN, _c.c_int, _c.POINTER(_c.c_char_p), _c.POINTER(_c.c_double), _I64P]
    L.nufft_strerror.argtypes = [_c.c_int]
    L.nufft_strerror.restype = _c.c_char_p
    L.nufft_last_cuda_error.restype = _c.c_int
    L.nufft_version.restype = _c.c_char_p
    _lib = L
    return L


def _strerror(code):
    try:
        return lib().nufft_strerror(int(code)).decode()
    except Exception:  # pragma: no cover
        return "?"


def version():
    return lib().nufft_version().decode()


def _check(code, what):
    if code != 0:
        extra = ""
        if code == -3:
            extra = " cudaError=%d" % lib().nufft_last_cuda_error()
        raise NufftError(code, what + extra)


def _dev(t, what, numel=None):
    """Device pointer of a contiguous complex64 CUDA tensor (no copies, no fallback)."""
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor (this library has no CPU path)" % what)
    if t.dtype != torch.complex64 or not t.is_contiguous():
        raise TypeError("%s must be a contiguous complex64 tensor" % what)
    if numel is not None and t.numel() != numel:
        raise ValueError("%s has %d elements, expected %d" % (what, t.numel(), numel))
    return _c.c_void_p(t.data_ptr())


def _stream():
    import torch
    return _c.c_void_p(torch.cuda.current_stream().cuda_stream)


class NufftPlan:
    """nufft_plan(Nd, Kd, Jd, om[M x d]) -> plan; methods mirror the C ABI on torch CUDA tensors.

    The host-buffer convenience calls (forward_host / adjoint_host) copy host arrays through pinned memory and are
    what bench.py's `e2e` leg times.
    """

    def __init__(self, Nd, Kd, Jd, om, max_batch=1, adjoint_mode=0, interp_mode=0, tile=None, max_subtile=0,
                 batch_layout=0, use_graphs=0, kernel="kb", coef_mode=0):
        L = lib()
        self.Nd = tuple(int(n) for n in Nd)
        self.Kd = tuple(int(k) for k in Kd)
        self.Jd = tuple(int(j) for j in Jd)
        d = len(self.Nd)
        om = np.ascontiguousarray(np.asarray(om, dtype=np.float64))
        if om.ndim != 2 or om.shape[1] != d:
            raise ValueError("om must be [M][d]")
        self.M = int(om.shape[0])
        self.d = d
        self.max_batch = int(max_batch)
        self.nimg = int(np.prod(self.Nd))
        self.cells = int(np.prod(self.Kd))
        opts = NufftOpts()
        _check(L.nufft_default_opts(_c.byref(opts)), "nufft_default_opts")
        opts.coef_mode = int(coef_mode)
        opts.adjoint_mode = int(adjoint_mode)
        opts.interp_mode = int(interp_mode)
        opts.max_subtile = int(max_subtile)
        opts.batch_layout = int(batch_layout)
        opts.use_graphs = int(use_graphs)
        opts.kernel = {"kb": 0, "minmax": 1}[kernel]
        if tile is not None:
            for a, t in enumerate(tile):
                opts.tile[a] = int(t)
        self._h = _PLAN()
        Nd_c = (_c.c_int64 * d)(*self.Nd)
        Kd_c = (_c.c_int64 * d)(*self.Kd)
        Jd_c = (_c.c_int * d)(*self.Jd)
        _check(L.nufft_plan(d, Nd_c, Kd_c, Jd_c, self.M, om.ctypes.data_as(_c.POINTER(_c.c_double)),
                            self.max_batch, _c.byref(opts), _c.byref(self._h)), "nufft_plan")
        self._coils = None

    # -- lifetime ---------------------------------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            import torch
            torch.cuda.synchronize()
            lib().nufft_destroy(self._h)
            self._h = _PLAN()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- helpers ----------------------------------------------------------------------------------------------
    def _batch_of(self, t, per):
        n = t.numel()
        if n % per != 0 or n == 0:
            raise ValueError("tensor size %d is not a multiple of %d" % (n, per))
        return n // per

    def _new(self, *shape):
        import torch
        return torch.empty(shape, dtype=torch.complex64, device="cuda")

    # -- transforms (C ABI names) -----------------------------------------------------------------------------
    def forward(self, x, y=None):
        b = self._batch_of(x, self.nimg)
        y = self._new(b, self.M) if y is None else y
        _check(lib().nufft_forward(self._h, b, _dev(x, "x"), _dev(y, "y", b * self.M) if self.M else None, _stream()),
               "nufft_forward")
        return y

    def adjoint(self, y, x=None):
        b = self._batch_of(y, self.M) if self.M else 1
        x = self._new(b, *self.Nd) if x is None else x
        _check(lib().nufft_adjoint(self._h, b, _dev(y, "y") if self.M else None, _dev(x, "x", b * self.nimg), _stream()),
               "nufft_adjoint")
        return x

    def adjoint_noalloc(self, y, x):
        """nufft_adjoint_noalloc: one image, caller-owned output, workspace in the library's static device array."""
        _check(lib().nufft_adjoint_noalloc(self._h, _dev(y, "y", self.M) if self.M else None, _dev(x, "x", self.nimg), _stream()),
               "nufft_adjoint_noalloc")
        return x

    def selfadjoint(self, x, out=None):
        b = self._batch_of(x, self.nimg)
        out = self._new(b, *self.Nd) if out is None else out
        _check(lib().nufft_selfadjoint(self._h, b, _dev(x, "x"), _dev(out, "out", b * self.nimg), _stream()),
               "nufft_selfadjoint")
        return out

    def stage_scale_fft(self, x, grid=None):
        b = self._batch_of(x, self.nimg)
        grid = self._new(b, *self.Kd) if grid is None else grid
        _check(lib().nufft_stage_scale_fft(self._h, b, _dev(x, "x"), _dev(grid, "grid", b * self.cells), _stream()),
               "nufft_stage_scale_fft")
        return grid

    def stage_interp(self, grid, y=None):
        b = self._batch_of(grid, self.cells)
        y = self._new(b, self.M) if y is None else y
        _check(lib().nufft_stage_interp(self._h, b, _dev(grid, "grid"), _dev(y, "y", b * self.M) if self.M else None,
                                        _stream()), "nufft_stage_interp")
        return y

    def stage_gridding(self, y, grid=None, batch=None):
        b = self._batch_of(y, self.M) if self.M else int(batch or 1)
        grid = self._new(b, *self.Kd) if grid is None else grid
        _check(lib().nufft_stage_gridding(self._h, b, _dev(y, "y") if self.M else None,
                                          _dev(grid, "grid", b * self.cells), _stream()), "nufft_stage_gridding")
        return grid

    def stage_fft_scale(self, grid, x=None):
        """x = S^H F^H grid.  NOTE: destroys `grid`."""
        b = self._batch_of(grid, self.cells)
        x = self._new(b, *self.Nd) if x is None else x
        _check(lib().nufft_stage_fft_scale(self._h, b, _dev(grid, "grid"), _dev(x, "x", b * self.nimg), _stream()),
               "nufft_stage_fft_scale")
        return x

    # -- multi-coil -------------------------------------------------------------------------------------------
    def set_coils(self, c):
        if c is None:
            _check(lib().nufft_set_coils(self._h, 0, None), "nufft_set_coils")
            self._coils = None
            return
        nc = self._batch_of(c, self.nimg)
        _check(lib().nufft_set_coils(self._h, nc, _dev(c, "coils")), "nufft_set_coils")
        self._coils = c          # keep the borrowed tensor alive
        self.ncoil = nc

    def forward_coils(self, x, y=None):
        y = self._new(self.ncoil, self.M) if y is None else y
        _check(lib().nufft_forward_coils(self._h, _dev(x, "x", self.nimg), _dev(y, "y", self.ncoil * self.M), _stream()),
               "nufft_forward_coils")
        return y

    def adjoint_coils(self, y, x=None):
        x = self._new(*self.Nd) if x is None else x
        _check(lib().nufft_adjoint_coils(self._h, _dev(y, "y", self.ncoil * self.M), _dev(x, "x", self.nimg), _stream()),
               "nufft_adjoint_coils")
        return x

    def selfadjoint_coils(self, x, out=None):
        out = self._new(*self.Nd) if out is None else out
        _check(lib().nufft_selfadjoint_coils(self._h, _dev(x, "x", self.nimg), _dev(out, "out", self.nimg), _stream()),
               "nufft_selfadjoint_coils")
        return out

    # -- "next" rows: density compensation, Toeplitz A^H A -------------------------------------------------------
    def density_weights(self, niter, w=None):
        w = self._new(self.M) if w is None else w
        _check(lib().nufft_density_weights(self._h, int(niter), _dev(w, "w", self.M), _stream()), "nufft_density_weights")
        return w

    def adjoint_dcf(self, y, w, x=None):
        b = self._batch_of(y, self.M)
        x = self._new(b, *self.Nd) if x is None else x
        _check(lib().nufft_adjoint_dcf(self._h, b, _dev(y, "y"), _dev(w, "w", self.M), _dev(x, "x", b * self.nimg),
                                       _stream()), "nufft_adjoint_dcf")
        return x

    def toeplitz_build(self, w=None):
        _check(lib().nufft_toeplitz_build(self._h, None if w is None else _dev(w, "w", self.M), _stream()),
               "nufft_toeplitz_build")

    def toeplitz_enable(self, on=True):
        _check(lib().nufft_toeplitz_enable(self._h, int(bool(on))), "nufft_toeplitz_enable")

    def selfadjoint_toeplitz(self, x, out=None):
        b = self._batch_of(x, self.nimg)
        out = self._new(b, *self.Nd) if out is None else out
        _check(lib().nufft_selfadjoint_toeplitz(self._h, b, _dev(x, "x"), _dev(out, "out", b * self.nimg), _stream()),
               "nufft_selfadjoint_toeplitz")
        return out

    def selfadjoint_toeplitz_coils(self, x, out=None):
        out = self._new(*self.Nd) if out is None else out
        _check(lib().nufft_selfadjoint_toeplitz_coils(self._h, _dev(x, "x", self.nimg), _dev(out, "out", self.nimg),
                                                      _stream()), "nufft_selfadjoint_toeplitz_coils")
        return out

    # -- solvers ----------------------------------------------------------------------------------------------
    def solve_cg(self, y, niter, use_coils=False, x=None, want_history=False):
        x = self._new(*self.Nd) if x is None else x
        hist = (_c.c_double * (niter + 1))() if want_history else None
        _check(lib().nufft_solve_cg(self._h, int(bool(use_coils)), _dev(y, "y"), _dev(x, "x", self.nimg), int(niter),
                                    hist, _stream()), "nufft_solve_cg")
        return (x, np.array(hist[:])) if want_history else x

    def solve_l1tv_ols(self, y, mu, lam, n_outer, n_inner, n_cg, use_coils=False, x=None):
        x = self._new(*self.Nd) if x is None else x
        _check(lib().nufft_solve_l1tv_ols(self._h, int(bool(use_coils)), _dev(y, "y"), _dev(x, "x", self.nimg),
                                          float(mu), float(lam), int(n_outer), int(n_inner), int(n_cg), _stream()),
               "nufft_solve_l1tv_ols")
        return x

    def solve_cg_kspace(self, y, niter, x=None, want_history=False):
        x = self._new(*self.Nd) if x is None else x
        hist = (_c.c_double * (niter + 1))() if want_history else None
        _check(lib().nufft_solve_cg_kspace(self._h, _dev(y, "y", self.M), _dev(x, "x", self.nimg), int(niter), hist,
                                           _stream()), "nufft_solve_cg_kspace")
        return (x, np.array(hist[:])) if want_history else x

    def solve_l1tv_lad(self, y, mu, lam, n_outer, n_inner, n_cg, use_coils=False, x=None):
        x = self._new(*self.Nd) if x is None else x
        _check(lib().nufft_solve_l1tv_lad(self._h, int(bool(use_coils)), _dev(y, "y"), _dev(x, "x", self.nimg),
                                          float(mu), float(lam), int(n_outer), int(n_inner), int(n_cg), _stream()),
               "nufft_solve_l1tv_lad")
        return x

    # -- info -------------------------------------------------------------------------------------------------
    def info(self):
        v = [_c.c_int64() for _ in range(5)]
        _check(lib().nufft_plan_info(self._h, *[_c.byref(a) for a in v]), "nufft_plan_info")
        keys = ["bytes_plan", "bytes_work", "n_tiles", "n_work", "max_tile_samples"]
        out = {k: int(a.value) for k, a in zip(keys, v)}
        J, kern, paths, perr = _c.c_int(), _c.c_int(), _c.c_int(), _c.c_double()
        _check(lib().nufft_plan_modes(self._h, _c.byref(J), _c.byref(kern), _c.byref(paths), _c.byref(perr)),
               "nufft_plan_modes")
        hist = (_c.c_int64 * 24)()
        _check(lib().nufft_plan_tile_histogram(self._h, hist), "nufft_plan_tile_histogram")
        out["tile_histogram"] = [int(v) for v in hist]
        out.update(J=J.value, kernel=("kb", "minmax")[kern.value], interleaved=bool(paths.value & 1),
                   caller_order_interp=bool(paths.value & 2), generic_width_kernels=bool(paths.value & 4),
                   toeplitz=bool(paths.value & 8), poly_err=perr.value)
        return out

    def launch_count(self):
        return int(lib().nufft_launch_count(self._h))

    def profile_enable(self, on=True):
        _check(lib().nufft_profile_enable(self._h, int(bool(on))), "nufft_profile_enable")

    def profile_reset(self):
        _check(lib().nufft_profile_reset(self._h), "nufft_profile_reset")

    def profile(self):
        """{kernel label: (total device ms, launches)} since the last reset (synchronises the recorded events)."""
        out = {}
        for i in range(lib().nufft_profile_count(self._h)):
            name, ms, n = _c.c_char_p(), _c.c_double(), _c.c_int64()
            _check(lib().nufft_profile_get(self._h, i, _c.byref(name), _c.byref(ms), _c.byref(n)), "nufft_profile_get")
            out[name.value.decode()] = (float(ms.value), int(n.value))
        return out

    # -- host-buffer transforms (the e2e path): marshalling only, the chunked copy/compute pipeline is in the library --
    @staticmethod
    def _hostptr(t, what, numel):
        import torch
        if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.complex64 or not t.is_contiguous():
            raise TypeError("%s must be a contiguous complex64 CPU tensor (pinned for overlap)" % what)
        if t.numel() != numel:
            raise ValueError("%s has %d elements, expected %d" % (what, t.numel(), numel))
        return _c.c_void_p(t.data_ptr())

    def _new_host(self, *shape):
        import torch
        return torch.empty(shape, dtype=torch.complex64, pin_memory=True)

    def host_input_ready(self, on=True):
        _check(lib().nufft_host_input_ready(self._h, int(bool(on))), "nufft_host_input_ready")

    def forward_host(self, x_host, y_host=None):
        """x_host: pinned CPU complex64 [b][Nd] -> y_host pinned CPU [b][M].  Asynchronous on the current stream."""
        b = self._batch_of(x_host, self.nimg)
        y_host = self._new_host(b, self.M) if y_host is None else y_host
        _check(lib().nufft_forward_host(self._h, b, self._hostptr(x_host, "x_host", b * self.nimg),
                                        self._hostptr(y_host, "y_host", b * self.M), _stream()), "nufft_forward_host")
        return y_host

    def adjoint_host(self, y_host, x_host=None):
        b = self._batch_of(y_host, self.M)
        x_host = self._new_host(b, *self.Nd) if x_host is None else x_host
        _check(lib().nufft_adjoint_host(self._h, b, self._hostptr(y_host, "y_host", b * self.M),
                                        self._hostptr(x_host, "x_host", b * self.nimg), _stream()), "nufft_adjoint_host")
        return x_host

    def selfadjoint_host(self, x_host, out_host=None):
        b = self._batch_of(x_host, self.nimg)
        out_host = self._new_host(b, *self.Nd) if out_host is None else out_host
        _check(lib().nufft_selfadjoint_host(self._h, b, self._hostptr(x_host, "x_host", b * self.nimg),
                                            self._hostptr(out_host, "out_host", b * self.nimg), _stream()),
               "nufft_selfadjoint_host")
        return out_host
