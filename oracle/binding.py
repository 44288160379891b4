"""ctypes binding of oracle/liboracle.so (the plain-C CPU oracle; test infrastructure).

Argument marshalling only -- every number is computed by dgpe_oracle.c.
Arrays are numpy, host memory, complex128 / float64, C-contiguous, shape (nx, ny, nz).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

IMAG, REAL = 0, 1
OK, ERR_ARG, ERR_NOMEM, ERR_NONFINITE = 0, -1, -3, -5

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, dp, ci, cd = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_double
        L.odgpe_create.restype = vp
        L.odgpe_create.argtypes = [ci, ci, ci, cd, cd, cd, cd, cd, cd, cd, cd, cd, ci]
        L.odgpe_destroy.restype = None
        L.odgpe_destroy.argtypes = [vp]
        L.odgpe_step.argtypes = [vp, vp, ci]
        for name in ("odgpe_norm", "odgpe_chempot", "odgpe_energy", "odgpe_rms", "odgpe_energy_terms"):
            getattr(L, name).argtypes = [vp, vp, dp]
        L.odgpe_dft1.argtypes = [ci, vp, ci]
        L.odgpe_dft3.argtypes = [ci, ci, ci, vp, ci]
        L.odgpe_dipolar.argtypes = [vp, vp, vp]
        L.odgpe_nonlinear.argtypes = [vp, vp]
        L.odgpe_sweep.argtypes = [vp, vp, ci]
        _lib = L
    return _lib


def _c128(a, shape=None):
    assert isinstance(a, np.ndarray) and a.dtype == np.complex128 and a.flags.c_contiguous
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a.ctypes.data_as(C.c_void_p)


class Oracle:
    """odgpe_* on host arrays. psi arrays are modified in place."""

    def __init__(self, nx, ny, nz, dx, dy, dz, dt, gamma, nu, lam, g, gdd, mode):
        self.shape = (nx, ny, nz)
        self.h = lib().odgpe_create(nx, ny, nz, dx, dy, dz, dt, gamma, nu, lam, g, gdd, mode)
        if not self.h:
            raise ValueError("odgpe_create rejected the arguments")

    def close(self):
        if self.h:
            lib().odgpe_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def step(self, psi, nsteps=1):
        return lib().odgpe_step(self.h, _c128(psi, self.shape), int(nsteps))

    def _scalar(self, fn, psi, n=1):
        out = (C.c_double * n)()
        rc = fn(self.h, _c128(psi, self.shape), out)
        if rc != OK:
            raise RuntimeError(f"oracle call failed: {rc}")
        return out[0] if n == 1 else [out[i] for i in range(n)]

    def norm(self, psi):
        return self._scalar(lib().odgpe_norm, psi)

    def chempot(self, psi):
        return self._scalar(lib().odgpe_chempot, psi)

    def energy(self, psi):
        return self._scalar(lib().odgpe_energy, psi)

    def rms(self, psi):
        return self._scalar(lib().odgpe_rms, psi, 4)

    def energy_terms(self, psi):
        return self._scalar(lib().odgpe_energy_terms, psi, 4)

    def dipolar(self, dens):
        assert dens.dtype == np.float64 and dens.flags.c_contiguous and dens.shape == self.shape
        phi = np.empty_like(dens)
        rc = lib().odgpe_dipolar(self.h, dens.ctypes.data_as(C.c_void_p), phi.ctypes.data_as(C.c_void_p))
        if rc != OK:
            raise RuntimeError(f"odgpe_dipolar failed: {rc}")
        return phi

    def nonlinear(self, psi):
        return lib().odgpe_nonlinear(self.h, _c128(psi, self.shape))

    def sweep(self, psi, axis):
        return lib().odgpe_sweep(self.h, _c128(psi, self.shape), int(axis))


def dft1(line, sign):
    a = np.ascontiguousarray(line, dtype=np.complex128).copy()
    rc = lib().odgpe_dft1(a.size, _c128(a), int(sign))
    assert rc == OK
    return a


def dft3(a, sign):
    a = np.ascontiguousarray(a, dtype=np.complex128).copy()
    nx, ny, nz = a.shape
    rc = lib().odgpe_dft3(nx, ny, nz, _c128(a), int(sign))
    assert rc == OK
    return a
