"""ctypes binding of libdgpe.so -- the C-ABI of include/dgpe.h, same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; there is no CPU fallback: if the built
library or a CUDA device is missing, the calls raise.  torch is used for device memory and streams.
"""
import ctypes as C
import os

import torch

from . import build as _build

IMAG, REAL, IMAG_RPSI = 0, 1, 2
OK, ERR_ARG, ERR_CUDA, ERR_NOMEM, ERR_UNSUPPORTED, ERR_NONFINITE = 0, -1, -2, -3, -4, -5

EXPORTS = ("dgpe_create", "dgpe_create_ex", "dgpe_last_error_code", "dgpe_destroy", "dgpe_set_stream", "dgpe_step", "dgpe_norm", "dgpe_chempot",
           "dgpe_energy", "dgpe_rms", "dgpe_energy_terms", "dgpe_dipolar", "dgpe_nonlinear", "dgpe_sweep",
           "dgpe_step_host", "dgpe_step_profile", "dgpe_kernel_name", "dgpe_kernel_bytes",
           "dgpe_synchronize", "dgpe_bytes_per_step", "dgpe_launches_per_step", "dgpe_last_error",
           # one rank's stages of the slab-decomposed step (bound in sharded.py)
           "dgpe_slab_create", "dgpe_slab_destroy", "dgpe_slab_set_stream", "dgpe_slab_elems", "dgpe_slab_begin",
           "dgpe_slab_stage_a", "dgpe_slab_stage_b", "dgpe_slab_stage_c", "dgpe_slab_stage_d", "dgpe_slab_stage_e",
           "dgpe_slab_end",
           # the norm without any allocation (static device scratch)
           "dgpe_norm_noalloc")

_lib = None

# fields of dgpe_options (include/dgpe.h), in order; -1 = the library's default
OPTION_FIELDS = ("generic", "tma", "tma_fft", "tma_k3", "graph", "prefetch", "pf_mult", "tma_pair")


class DgpeOptions(C.Structure):
    _fields_ = [(name, C.c_int) for name in OPTION_FIELDS] + [("reserved", C.c_int * 8)]

    def __init__(self, **kw):
        super().__init__()
        for name in OPTION_FIELDS:
            setattr(self, name, -1)
        for i in range(8):
            self.reserved[i] = -1
        for name, val in kw.items():
            if name not in OPTION_FIELDS:
                raise KeyError(f"unknown dgpe option {name!r} (known: {OPTION_FIELDS})")
            setattr(self, name, int(val))


def parse_options(text):
    """'generic=1,tma=0' -> dict, for command lines (bench.py --opt); the library reads no environment."""
    out = {}
    for item in (text or "").split(","):
        if item.strip():
            k, _, v = item.partition("=")
            out[k.strip()] = int(v)
    return out


class DgpeError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"dgpe error {code}: {msg}")
        self.code = code


def lib():
    """Load (building if needed) paper_1610_05329_b200/libdgpe.so.  Raises if it cannot be built/loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, dp, ci, cd = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_double
        L.dgpe_create.restype = vp
        L.dgpe_create.argtypes = [ci, ci, ci, cd, cd, cd, cd, cd, cd, cd, cd, cd, ci]
        L.dgpe_create_ex.restype = vp
        L.dgpe_create_ex.argtypes = [ci, ci, ci, cd, cd, cd, cd, cd, cd, cd, cd, cd, ci, C.POINTER(DgpeOptions)]
        L.dgpe_last_error_code.restype = ci
        L.dgpe_last_error_code.argtypes = []
        L.dgpe_destroy.restype = None
        L.dgpe_destroy.argtypes = [vp]
        L.dgpe_set_stream.argtypes = [vp, vp]
        L.dgpe_step.argtypes = [vp, vp, ci]
        for name in ("dgpe_norm", "dgpe_chempot", "dgpe_energy", "dgpe_rms", "dgpe_energy_terms"):
            getattr(L, name).argtypes = [vp, vp, dp]
        L.dgpe_dipolar.argtypes = [vp, vp, vp]
        L.dgpe_nonlinear.argtypes = [vp, vp]
        L.dgpe_sweep.argtypes = [vp, vp, ci]
        L.dgpe_step_host.argtypes = [vp, vp, ci]
        L.dgpe_step_profile.argtypes = [vp, vp, ci, dp]
        L.dgpe_kernel_name.restype = C.c_char_p
        L.dgpe_kernel_name.argtypes = [vp, ci]
        L.dgpe_kernel_bytes.restype = cd
        L.dgpe_kernel_bytes.argtypes = [vp, ci]
        L.dgpe_synchronize.argtypes = [vp]
        L.dgpe_bytes_per_step.restype = cd
        L.dgpe_bytes_per_step.argtypes = [vp]
        L.dgpe_launches_per_step.argtypes = [vp]
        L.dgpe_norm_noalloc.argtypes = [vp, ci, ci, ci, cd, cd, cd, vp, vp]
        L.dgpe_last_error.restype = C.c_char_p
        L.dgpe_last_error.argtypes = []
        _lib = L
    return _lib


def last_error():
    return lib().dgpe_last_error().decode()


def _check(rc):
    if rc != OK:
        raise DgpeError(rc, last_error())


NOALLOC_MAX_NX = 1024


def norm_noalloc(psi, dx, dy, dz, out, stream=None):
    """dgpe_norm_noalloc: out (CUDA float64 tensor, one element, caller-owned) <- sum |psi|^2 dx dy dz, asynchronously on
    `stream` (default: torch's current stream).  Allocates nothing, needs no handle; nx <= NOALLOC_MAX_NX.  Calls that
    overlap on the GPU race on the library's static scratch: keep them on one stream.  Returns the status code."""
    if not (isinstance(psi, torch.Tensor) and psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.dim() == 3):
        raise TypeError("psi must be a contiguous 3-D CUDA complex128 tensor")
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.numel() == 1
            and out.device == psi.device):
        raise TypeError("out must be a one-element CUDA float64 tensor on psi's device")
    st = stream if stream is not None else torch.cuda.current_stream(psi.device)
    ptr = st.cuda_stream if hasattr(st, "cuda_stream") else int(st or 0)
    nx, ny, nz = psi.shape
    with torch.cuda.device(psi.device):
        return lib().dgpe_norm_noalloc(C.c_void_p(psi.data_ptr()), nx, ny, nz, dx, dy, dz, C.c_void_p(out.data_ptr()),
                                       C.c_void_p(ptr))


class Dgpe:
    """One dgpe_handle.  psi arguments are contiguous torch.complex128 CUDA tensors of shape (nx, ny, nz)
    (torch.float64 for mode IMAG_RPSI, the real-valued imaginary-time path)."""

    def __init__(self, nx, ny, nz, dx, dy, dz, dt, gamma, nu, lam, g, gdd, mode, stream=None, options=None):
        """options: dict of dgpe_options fields (kernel selection for A/B runs and cross-checks) -> dgpe_create_ex."""
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1610_05329_b200 needs a CUDA device (no CPU fallback)")
        self.shape = (nx, ny, nz)
        self.mode = mode
        self.dtype = torch.float64 if mode == IMAG_RPSI else torch.complex128
        self.device = torch.device("cuda", torch.cuda.current_device())
        if options:
            opt = DgpeOptions(**options)
            self.h = lib().dgpe_create_ex(nx, ny, nz, dx, dy, dz, dt, gamma, nu, lam, g, gdd, mode, C.byref(opt))
        else:
            self.h = lib().dgpe_create(nx, ny, nz, dx, dy, dz, dt, gamma, nu, lam, g, gdd, mode)
        if not self.h:
            raise DgpeError(lib().dgpe_last_error_code() or ERR_ARG, last_error())
        self.set_stream(stream if stream is not None else torch.cuda.current_stream())

    def close(self):
        if getattr(self, "h", None):
            lib().dgpe_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream):
        ptr = stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream or 0)
        _check(lib().dgpe_set_stream(self.h, C.c_void_p(ptr)))

    def _psi(self, psi):
        if not (isinstance(psi, torch.Tensor) and psi.is_cuda and psi.dtype == self.dtype
                and psi.is_contiguous() and tuple(psi.shape) == self.shape):
            raise TypeError(f"psi must be a contiguous CUDA {self.dtype} tensor of shape {self.shape}")
        if psi.device != self.device:
            raise TypeError(f"psi lives on {psi.device} but the handle was created on {self.device}")
        return C.c_void_p(psi.data_ptr())

    def step(self, psi, nsteps=1):
        """dgpe_step; returns the status code (OK or ERR_NONFINITE), raises on every other error."""
        rc = lib().dgpe_step(self.h, self._psi(psi), int(nsteps))
        if rc not in (OK, ERR_NONFINITE):
            _check(rc)
        return rc

    def step_host(self, psi_host, nsteps=1):
        """dgpe_step_host on a contiguous CPU tensor of the handle's dtype (pinned for full-speed copies)."""
        if not (isinstance(psi_host, torch.Tensor) and not psi_host.is_cuda and psi_host.dtype == self.dtype
                and psi_host.is_contiguous() and tuple(psi_host.shape) == self.shape):
            raise TypeError(f"psi_host must be a contiguous CPU {self.dtype} tensor of shape {self.shape}")
        rc = lib().dgpe_step_host(self.h, C.c_void_p(psi_host.data_ptr()), int(nsteps))
        if rc not in (OK, ERR_NONFINITE):
            _check(rc)
        return rc

    def step_profile(self, psi, nsteps=1):
        """dgpe_step_profile: list of (kernel name, algorithmic bytes, average ms) for the kernels of a step."""
        nk = self.launches_per_step
        ms = (C.c_double * nk)()
        rc = lib().dgpe_step_profile(self.h, self._psi(psi), int(nsteps), ms)
        if rc not in (OK, ERR_NONFINITE):
            _check(rc)
        return [(lib().dgpe_kernel_name(self.h, k).decode(), lib().dgpe_kernel_bytes(self.h, k), ms[k])
                for k in range(nk)]

    def _scalars(self, fn, psi, n):
        out = (C.c_double * n)()
        _check(fn(self.h, self._psi(psi), out))
        return out[0] if n == 1 else [out[i] for i in range(n)]

    def norm(self, psi):
        return self._scalars(lib().dgpe_norm, psi, 1)

    def chempot(self, psi):
        return self._scalars(lib().dgpe_chempot, psi, 1)

    def energy(self, psi):
        return self._scalars(lib().dgpe_energy, psi, 1)

    def rms(self, psi):
        return self._scalars(lib().dgpe_rms, psi, 4)

    def energy_terms(self, psi):
        return self._scalars(lib().dgpe_energy_terms, psi, 4)

    def dipolar(self, psi):
        phi = torch.empty(self.shape, dtype=torch.float64, device=psi.device)
        _check(lib().dgpe_dipolar(self.h, self._psi(psi), C.c_void_p(phi.data_ptr())))
        return phi

    def nonlinear(self, psi):
        _check(lib().dgpe_nonlinear(self.h, self._psi(psi)))

    def sweep(self, psi, axis):
        _check(lib().dgpe_sweep(self.h, self._psi(psi), int(axis)))

    def synchronize(self):
        _check(lib().dgpe_synchronize(self.h))

    @property
    def bytes_per_step(self):
        return lib().dgpe_bytes_per_step(self.h)

    @property
    def launches_per_step(self):
        return lib().dgpe_launches_per_step(self.h)
