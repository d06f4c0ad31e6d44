"""Helpers shared by the GPU parity tests (no method arithmetic of their own beyond calling oracle/)."""
import numpy as np

from oracle import nufft_oracle as orc


def rel(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def noisy_density_weights(om, Nd, Kd, Jd, niter, eps, seed=0):
    """The oracle's density-compensation iteration (eq. (6), reading R21) with relative noise eps injected after every
    operator application: what ANY implementation whose operators agree with the oracle to eps must expect (the iteration
    divides by |A A^H w|, which amplifies perturbations where that magnitude is small)."""
    rng = np.random.default_rng(seed)

    def noisy(v):
        n = np.linalg.norm(v) / np.sqrt(v.size)
        return v + eps * n * (rng.standard_normal(v.shape) + 1j * rng.standard_normal(v.shape))

    w = np.ones(om.shape[0])
    for _ in range(niter):
        t = noisy(orc.forward(noisy(orc.adjoint(w.astype(np.complex128), om, Nd, Kd, Jd)), om, Nd, Kd, Jd))
        w = w / np.abs(t)
    return w


def check_density_weights(wg, wo, om, Nd, Kd, Jd, niter, tol):
    """w itself against the oracle: <= tol, or within 3x of what the float64 oracle moves by when its operators carry the
    GPU's own 2e-7 relative rounding (max over three seeds); and |A A^H w| = w_prev / w to tol where that is defined."""
    err = rel(wg, wo)
    floor = max(rel(noisy_density_weights(om, Nd, Kd, Jd, niter, 2e-7, seed=s), wo) for s in (0, 1, 2))
    assert np.all(np.isfinite(wg)) and err < max(tol, 3.0 * floor), (err, floor)
    return err, floor


def coil_ops_threaded(c128, om, Nd, Kd, Jd, with_forward=False):
    """A_multi^H A_multi and A_multi^H of the oracle, the per-coil transforms (oracle/nufft_oracle.py forward / adjoint,
    unchanged) evaluated on a thread pool: same arithmetic, same fixed summation order over the coils."""
    import concurrent.futures as cf
    import os
    pool = cf.ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1))

    def AHy(y):
        parts = list(pool.map(lambda i: np.conj(c128[i]) * orc.adjoint(y[i], om, Nd, Kd, Jd), range(len(c128))))
        out = np.zeros(tuple(Nd), dtype=np.complex128)
        for q in parts:
            out += q
        return out

    def AHA(z):
        parts = list(pool.map(lambda i: np.conj(c128[i]) * orc.adjoint(orc.forward(c128[i] * z, om, Nd, Kd, Jd), om, Nd, Kd, Jd),
                              range(len(c128))))
        out = np.zeros(tuple(Nd), dtype=np.complex128)
        for q in parts:
            out += q
        return out

    def A(z):
        return np.stack(list(pool.map(lambda i: orc.forward(c128[i] * z, om, Nd, Kd, Jd), range(len(c128)))))
    return (AHA, AHy, A) if with_forward else (AHA, AHy)
