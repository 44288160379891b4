"""Slab-decomposed SSCN step over several GPUs.

The paper's MPI packages distribute psi "along NX": rank p owns the x slab psi[p NX/P:(p+1) NX/P][NY][NZ].  The y and z
passes and sweeps are local; the x pass of the dipolar convolution and the x sweep need "the whole NX extent" and therefore run
after an all-to-all that leaves the data "locally transposed", NX x (NY/P) x NZ, every rank sending every peer one
(NX/P) x (NY/P) x NZ block, and are followed by the exchange back: four all-to-alls per step (two of the half-spectrum,
two of psi) and one all-reduce of a double (the norm, imaginary time).

Every local stage runs in the CUDA library (dgpe_slab_* of include/dgpe.h: the same kernels as dgpe_step, launched on slab
views); this module only sequences the stages and hands the blocks to a communicator:

  DistComm   one rank per process and GPU: torch.distributed (backend "nccl" over NVLink / NVSwitch; "gloo" for CPU tensors in the
             tests of the exchange itself).
  LocalComm  all ranks are emulated inside one process on ONE device: the exchange is a set of device-to-device copies.  This is
             how the sharded path is checked element by element against the oracle on the single GPU this build can reach.

What the paper found (the transposes dominate, no speed-up below 4 nodes) is expected here too: an all-to-all moves
16N/P (or S/P) bytes per rank over NVLink at ~0.77 TB/s measured per direction, against 6.5 TB/s for a local pass over the same
bytes.  UNMEASURED on hardware: no multi-GPU node was available to this build.
"""
import ctypes as C

import torch

from . import binding as _b

IMAG, REAL = _b.IMAG, _b.REAL


def block_elems(nx, ny, w, nranks):
    """Elements of the block one rank sends to one peer: (NX/P) x (NY/P) x w."""
    if nx % nranks or ny % nranks:
        raise ValueError(f"nx = {nx} and ny = {ny} must both be divisible by the number of ranks {nranks} (P:L132)")
    return (nx // nranks) * (ny // nranks) * w


def _lib():
    L = _b.lib()
    if not getattr(L, "_slab_ready", False):
        vp, ci, cd = C.c_void_p, C.c_int, C.c_double
        L.dgpe_slab_create.restype = vp
        L.dgpe_slab_create.argtypes = [ci, ci, ci, cd, cd, cd, cd, cd, cd, cd, cd, cd, ci, ci, ci]
        L.dgpe_slab_destroy.restype = None
        L.dgpe_slab_destroy.argtypes = [vp]
        L.dgpe_slab_set_stream.argtypes = [vp, vp]
        L.dgpe_slab_elems.restype = C.c_longlong
        L.dgpe_slab_elems.argtypes = [vp, ci]
        L.dgpe_slab_begin.argtypes = [vp]
        L.dgpe_slab_stage_a.argtypes = [vp, vp, vp]
        L.dgpe_slab_stage_b.argtypes = [vp, vp]
        L.dgpe_slab_stage_c.argtypes = [vp, vp, vp, vp]
        L.dgpe_slab_stage_d.argtypes = [vp, vp, vp]
        L.dgpe_slab_stage_e.argtypes = [vp, vp, vp, vp]
        L.dgpe_slab_end.argtypes = [vp, vp]
        L._slab_ready = True
    return L


# ------------------------------------------------------------------------------------------------
# communicators: all_to_all over equal blocks in rank order, and the sum of one double per rank
# ------------------------------------------------------------------------------------------------
class DistComm:
    """One local rank; the peers are the other processes of a torch.distributed group."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.world = dist.get_world_size(group)
        self.rank = dist.get_rank(group)
        self.local_ranks = [self.rank]

    def all_to_all(self, send, recv):
        """send[0], recv[0]: flat tensors of world equal blocks; block q of send goes to rank q, block p of recv comes from p."""
        s, r = send[0], recv[0]
        if s.is_complex():                       # NCCL moves bytes: exchange the (re, im) pairs as doubles
            s, r = torch.view_as_real(s).reshape(-1), torch.view_as_real(r).reshape(-1)
        self.dist.all_to_all_single(r, s, group=self.group)

    def all_reduce_sum(self, vals):
        self.dist.all_reduce(vals[0], op=self.dist.ReduceOp.SUM, group=self.group)


class LocalComm:
    """All `world` ranks live in this process on one device (emulation): block q of rank p's send buffer is copied to
    block p of rank q's receive buffer; the norm parts are added in rank order (deterministic)."""

    def __init__(self, world):
        self.world = world
        self.rank = 0
        self.local_ranks = list(range(world))

    def all_to_all(self, send, recv):
        P = self.world
        for q in range(P):
            rq = recv[q].view(P, -1)
            for p in range(P):
                rq[p].copy_(send[p].view(P, -1)[q])

    def all_reduce_sum(self, vals):
        tot = vals[0].clone()
        for v in vals[1:]:
            tot += v
        for v in vals:
            v.copy_(tot)


# ------------------------------------------------------------------------------------------------
class ShardedDgpe:
    """The sharded step for the ranks that live in this process (one with DistComm, all with LocalComm).

    psi_slabs: one contiguous complex128 CUDA tensor (nx/P, ny, nz) per local rank -- rank p's x slab -- advanced in place."""

    def __init__(self, nx, ny, nz, dx, dy, dz, dt, gamma, nu, lam, g, gdd, mode, comm):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1610_05329_b200 needs a CUDA device (no CPU fallback)")
        if mode not in (IMAG, REAL):
            raise ValueError("the sharded step takes DGPE_IMAG or DGPE_REAL")
        self.comm, self.mode, self.P = comm, mode, comm.world
        self.shape = (nx, ny, nz)
        self.slab_shape = (nx // self.P, ny, nz)
        block_elems(nx, ny, nz, self.P)          # divisibility
        L = _lib()
        self.h = []
        for r in comm.local_ranks:
            h = L.dgpe_slab_create(nx, ny, nz, dx, dy, dz, dt, gamma, nu, lam, g, gdd, mode, self.P, r)
            if not h:
                raise _b.DgpeError(L.dgpe_last_error_code() or _b.ERR_ARG, _b.last_error())
            self.h.append(h)
            _b._check(L.dgpe_slab_set_stream(h, C.c_void_p(torch.cuda.current_stream().cuda_stream)))
        ns, npsi = L.dgpe_slab_elems(self.h[0], 1), L.dgpe_slab_elems(self.h[0], 0)
        dev = torch.device("cuda", torch.cuda.current_device())
        mk = lambda n, dt_: [torch.empty(n, dtype=dt_, device=dev) for _ in self.h]
        # two buffers per kind and rank: what leaves and what arrives (the arriving one is the y slab)
        self.spec_a, self.spec_b = mk(ns, torch.complex128), mk(ns, torch.complex128)
        self.psi_a, self.psi_b = mk(npsi, torch.complex128), mk(npsi, torch.complex128)
        self.norm = mk(1, torch.float64)

    def close(self):
        for h in self.h:
            _lib().dgpe_slab_destroy(h)
        self.h = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ptr(self, t):
        return C.c_void_p(t.data_ptr())

    def step(self, psi_slabs, nsteps=1):
        """Advance every local slab by nsteps steps; returns the status (OK or ERR_NONFINITE)."""
        L, H = _lib(), self.h
        if len(psi_slabs) != len(H):
            raise ValueError("one psi slab per local rank")
        for t in psi_slabs:
            if not (t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous() and tuple(t.shape) == self.slab_shape):
                raise TypeError(f"psi slabs must be contiguous CUDA complex128 tensors of shape {self.slab_shape}")
        if nsteps <= 0:
            return _b.OK
        imag = self.mode == IMAG
        for h in H:
            _b._check(L.dgpe_slab_begin(h))
        for _ in range(nsteps):
            for h, psi, sa in zip(H, psi_slabs, self.spec_a):
                _b._check(L.dgpe_slab_stage_a(h, self._ptr(psi), self._ptr(sa)))
            self.comm.all_to_all(self.spec_a, self.spec_b)                    # x slabs -> y slabs
            for h, sb in zip(H, self.spec_b):
                _b._check(L.dgpe_slab_stage_b(h, self._ptr(sb)))
            self.comm.all_to_all(self.spec_b, self.spec_a)                    # and back
            for h, psi, sa, pa in zip(H, psi_slabs, self.spec_a, self.psi_a):
                _b._check(L.dgpe_slab_stage_c(h, self._ptr(sa), self._ptr(psi), self._ptr(pa)))
            self.comm.all_to_all(self.psi_a, self.psi_b)                      # psi: x slabs -> y slabs
            for h, pb, nr in zip(H, self.psi_b, self.norm):
                _b._check(L.dgpe_slab_stage_d(h, self._ptr(pb), self._ptr(nr) if imag else None))
            self.comm.all_to_all(self.psi_b, self.psi_a)                      # and back
            if imag:
                self.comm.all_reduce_sum(self.norm)
            for h, psi, pa, nr in zip(H, psi_slabs, self.psi_a, self.norm):
                _b._check(L.dgpe_slab_stage_e(h, self._ptr(pa), self._ptr(psi), self._ptr(nr) if imag else None))
        status = _b.OK
        for h, psi in zip(H, psi_slabs):
            rc = L.dgpe_slab_end(h, self._ptr(psi))
            if rc not in (_b.OK, _b.ERR_NONFINITE):
                _b._check(rc)
            status = status or rc
        return status
