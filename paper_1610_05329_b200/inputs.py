"""Seeded synthetic inputs for the dipolar-GPE SSCN step (configs C1..C5 of BASELINE.json).

This module serves BOTH the CUDA library and the CPU oracle and therefore holds none of the
method's arithmetic: only the grid/physics parameters of each config, a counter-based random
number generator, and the initial wave functions (Gaussians, seeded noise, seeded phase field,
zeroed faces, unit norm).  Recipe: DESIGN.md section 5.

The paper times its programs on 480^3-class grids with physical parameters it does not state
 and on no public data set; BASELINE.json's configs stand in for that
workload: one trapped, smooth, Gaussian-like cloud in the middle of a box with Dirichlet
walls far away, complex fp64.
"""
from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import numpy as np

IMAG, REAL = 0, 1


@dataclass(frozen=True)
class Config:
    name: str
    shape: Tuple[int, int, int]
    d: Tuple[float, float, float]
    dt: float
    trap: Tuple[float, float, float]          # gamma, nu, lambda
    g: float
    gdd: float
    mode: int
    nsteps: int
    seed: int
    gauss: Tuple[float, float, float]         # psi0 ~ exp(-(a x^2 + b y^2 + c z^2)/2)
    noise: float = 1e-3
    phase_waves: int = 0                      # C5: number of random plane waves in the phase
    phase_amp: float = 0.1
    # C3 only: imaginary-time relaxation that precedes the real-time run
    relax: Optional["Config"] = field(default=None, compare=False)

    def create_args(self):
        """Positional arguments of dgpe_create / odgpe_create."""
        nx, ny, nz = self.shape
        return (nx, ny, nz, *self.d, self.dt, *self.trap, self.g, self.gdd, self.mode)

    @property
    def npoints(self):
        return self.shape[0] * self.shape[1] * self.shape[2]


def _c3():
    relax = Config("C3-relax", (256,) * 3, (0.15,) * 3, 0.001, (1.0, 1.0, 2.0), 80.0, 40.0, IMAG, 300, 3,
                   (1.0, 1.0, 2.0))
    return Config("C3", (256,) * 3, (0.15,) * 3, 0.001, (1.0, 1.0, 2.0), 64.0, 40.0, REAL, 1000, 3,
                  (1.0, 1.0, 2.0), relax=relax)


CONFIGS = {
    # BJ:configs[0]
    "C1": Config("C1", (64,) * 3, (0.25,) * 3, 0.005, (1.0, 1.0, 1.0), 20.0, 5.0, IMAG, 100, 1, (1.0, 1.0, 1.0)),
    # BJ:configs[1]
    "C2": Config("C2", (128,) * 3, (0.2,) * 3, 0.004, (0.5, 0.5, 1.0), 60.0, 30.0, IMAG, 500, 2, (0.5, 0.5, 1.0)),
    # BJ:configs[2]
    "C3": _c3(),
    # BJ:configs[3]  (headline)
    "C4": Config("C4", (512,) * 3, (0.1,) * 3, 0.002, (1.0, 1.0, 4.0), 300.0, 200.0, IMAG, 200, 4, (1.0, 1.0, 4.0)),
    # BJ:configs[4]
    "C5": Config("C5", (768, 768, 384), (0.1, 0.1, 0.2), 0.001, (0.25, 0.25, 1.0), 500.0, 450.0, REAL, 200, 5,
                 (0.25, 0.25, 1.0), phase_waves=8),
}


# The grids of the paper's own timing tables (Table 1: 480^3; Table 2: 480x480x500; P:L111
# Table 3: 480x480x250), for like-for-like CONTEXT runs only (`bench.py --config T1i` ...).  The paper
# does not state the physics of those runs, so they borrow C4's spacings, time step, trap
# and interaction strengths; timing is data-independent.  i = imaginary time, r = real time.
PAPER_GRIDS = {"T1": (480, 480, 480), "T2": (480, 480, 500), "T3": (480, 480, 250)}
for _k, _shape in PAPER_GRIDS.items():
    for _m, _mode in (("i", IMAG), ("r", REAL)):
        CONFIGS[_k + _m] = Config(_k + _m, _shape, (0.1,) * 3, 0.002, (1.0, 1.0, 4.0), 300.0, 200.0, _mode, 1000, 4,
                                  (1.0, 1.0, 4.0))


def scaled(cfg: Config, shape, name=None) -> Config:
    """Same physics on a smaller grid (same spacings): for parity cases the oracle finishes quickly."""
    return replace(cfg, shape=tuple(shape), name=name or f"{cfg.name}@{'x'.join(map(str, shape))}",
                   relax=None if cfg.relax is None else replace(cfg.relax, shape=tuple(shape)))


# ---------------------------------------------------------------------------------------------
# counter-based generator: value depends only on (seed, stream, counter), not on generation order
# ---------------------------------------------------------------------------------------------

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    z = z.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        z ^= z >> np.uint64(30)
        z *= np.uint64(0xBF58476D1CE4E5B9)
        z ^= z >> np.uint64(27)
        z *= np.uint64(0x94D049BB133111EB)
        z ^= z >> np.uint64(31)
    return z


def uniform01(seed: int, stream: int, counter: np.ndarray) -> np.ndarray:
    """U[0,1) doubles keyed by (seed, stream, counter)."""
    with np.errstate(over="ignore"):
        key = _mix64(np.asarray([(seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03) & 0xFFFFFFFFFFFFFFFF],
                                dtype=np.uint64))[0]
        z = _mix64(counter.astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15) + key)
        z = _mix64(z ^ key)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def coords(n: int, d: float) -> np.ndarray:
    """Grid coordinates x_i = (i - n/2) d  (the box [-n d/2, n d/2))."""
    return (np.arange(n, dtype=np.float64) - n // 2) * d


def initial_state(cfg: Config) -> np.ndarray:
    """psi0 (complex128, shape cfg.shape): Gaussian x (1 + noise*U(-1,1)) [x seeded phase field],
    six faces zeroed, then scaled to unit norm  sum |psi|^2 dV = 1."""
    nx, ny, nz = cfg.shape
    dx, dy, dz = cfg.d
    x, y, z = coords(nx, dx), coords(ny, dy), coords(nz, dz)
    a, b, c = cfg.gauss
    gy = np.exp(-0.5 * b * y * y)[:, None]
    gz = np.exp(-0.5 * c * z * z)[None, :]

    waves = None
    if cfg.phase_waves:
        m = cfg.phase_waves
        cnt = np.arange(4 * m, dtype=np.uint64)
        u = uniform01(cfg.seed, 1, cnt).reshape(m, 4)
        ints = np.floor(u[:, :3] * 9.0).astype(np.int64) - 4          # uniform on [-4, 4]
        for r in range(m):                                             # exclude the zero vector
            if not ints[r].any():
                ints[r, 2] = 1
        phases = 2.0 * np.pi * u[:, 3]
        q = 2.0 * np.pi * ints / np.array([nx * dx, ny * dy, nz * dz])
        waves = (q, phases)

    psi = np.empty((nx, ny, nz), dtype=np.complex128)
    plane = ny * nz
    jk = np.arange(plane, dtype=np.uint64).reshape(ny, nz)
    for i in range(nx):
        u = uniform01(cfg.seed, 0, np.uint64(i) * np.uint64(plane) + jk)
        amp = np.exp(-0.5 * a * x[i] * x[i]) * gy * gz * (1.0 + cfg.noise * (2.0 * u - 1.0))
        if waves is None:
            psi[i] = amp
        else:
            q, phases = waves
            s = np.zeros((ny, nz))
            for r in range(q.shape[0]):
                s += np.cos(q[r, 0] * x[i] + q[r, 1] * y[:, None] + q[r, 2] * z[None, :] + phases[r])
            psi[i] = amp * np.exp(1j * cfg.phase_amp * s)
    psi[0] = 0.0
    psi[-1] = 0.0
    psi[:, 0] = 0.0
    psi[:, -1] = 0.0
    psi[:, :, 0] = 0.0
    psi[:, :, -1] = 0.0
    nrm = 0.0
    for i in range(nx):
        nrm += float(np.sum(psi[i].real ** 2 + psi[i].imag ** 2))
    psi *= 1.0 / np.sqrt(nrm * dx * dy * dz)
    return psi


def random_state(shape, seed: int, zero_faces: bool = True) -> np.ndarray:
    """Unstructured complex test field (for stage-level parity cases), O(1) magnitude."""
    nx, ny, nz = shape
    cnt = np.arange(nx * ny * nz, dtype=np.uint64)
    re = 2.0 * uniform01(seed, 10, cnt) - 1.0
    im = 2.0 * uniform01(seed, 11, cnt) - 1.0
    psi = (re + 1j * im).reshape(shape)
    if zero_faces:
        psi[0] = psi[-1] = 0.0
        psi[:, 0] = psi[:, -1] = 0.0
        psi[:, :, 0] = psi[:, :, -1] = 0.0
    return np.ascontiguousarray(psi)
