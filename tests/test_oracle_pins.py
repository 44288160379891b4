"""Pins of the CPU oracle against what the paper / BASELINE.json and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: each expected value is a
brute-force definition on a tiny input, a closed form, an invariant, a library routine the oracle
does not use (numpy.fft, numpy.linalg), or a printed value under tests/golden/ (with its citation).
Pin numbers P1..P13 follow SURVEY.md section 8(c) / DESIGN.md section 4.
"""
import math
import os
from dataclasses import replace

import numpy as np
import pytest

from paper_1610_05329_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")
IMAG, REAL = 0, 1


def read_golden(name):
    out = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 3:
                out[(int(line[0]), line[1])] = float(line[2])
            elif len(line) == 2:
                out[line[0]] = float(line[1])
    return out


def brute_dft3(a, sign):
    """O(n^2) per axis: X = sum_j x_j exp(sign 2 pi i j k / n), straight from the definition."""
    out = a.astype(np.complex128)
    for ax, n in enumerate(a.shape):
        j = np.arange(n)
        W = np.exp(sign * 2j * np.pi * np.outer(j, j) / n)
        out = np.moveaxis(np.tensordot(W, out, axes=([1], [ax])), 0, ax)
    return out


def rand_c(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


# ------------------------------------------------------------------------------------------
# P1 / P2 / P3: the oracle's FFT is the DFT
# ------------------------------------------------------------------------------------------

@pytest.mark.parametrize("shape", [(8, 8, 8), (4, 8, 16),            # P1: radix 2 (BJ:north_star check 1)
                                   (6, 6, 6), (12, 6, 3), (9, 4, 6),  # P2: radix 3 and mixed
                                   (5, 7, 10), (11, 13, 22)])         # the other primes of P:L130
@pytest.mark.parametrize("sign", [-1, 1])
def test_p1_p2_dft3_is_brute_force_dft(oracle, shape, sign):
    a = rand_c(shape, 7)
    got = oracle.dft3(a, sign)
    ref = brute_dft3(a, sign)
    assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))


@pytest.mark.parametrize("n", [1, 2, 3, 4, 6, 8, 9, 12, 27, 64, 96, 384, 768, 480, 500, 250, 143, 572, 1001])
def test_p1_dft1_sizes(oracle, n):
    a = rand_c((n,), n)
    j = np.arange(n)
    for sign in (-1, 1):
        ref = np.exp(sign * 2j * np.pi * np.outer(j, j) / n) @ a
        assert np.max(np.abs(oracle.dft1(a, sign) - ref)) <= 1e-11 * max(1.0, np.max(np.abs(ref)))


def test_p3_real_input_hermitian_and_parseval(oracle):
    rng = np.random.default_rng(3)
    n = rng.standard_normal((6, 8, 12))
    X = oracle.dft3(n.astype(np.complex128), -1)
    # Hermitian symmetry of the spectrum of a real field
    idx = [(-np.arange(s)) % s for s in n.shape]
    Xm = X[np.ix_(*idx)]
    assert np.max(np.abs(X - np.conj(Xm))) <= 1e-12
    # Parseval
    assert abs(np.sum(np.abs(X) ** 2) / n.size - np.sum(n * n)) <= 1e-10
    # library routine the oracle does not use
    assert np.max(np.abs(X - np.fft.fftn(n))) <= 1e-11
    # inverse(forward) = N * identity
    back = oracle.dft3(X, +1) / n.size
    assert np.max(np.abs(back - n)) <= 1e-12


# ------------------------------------------------------------------------------------------
# P4 / P5 / P6: dipolar mean field
# ------------------------------------------------------------------------------------------

def make(oracle, shape, d, dt=0.01, trap=(1.0, 1.0, 1.0), g=0.0, gdd=1.0, mode=IMAG):
    return oracle.Oracle(*shape, *d, dt, *trap, g, gdd, mode)


def test_p4_plane_wave_closed_form(oracle):
    """n = 1 + a cos(q.r) with q a grid wave vector  =>  Phi = Udd(q) a cos(q.r) exactly;
    pins the k-grid, the axis <-> kz assignment (dipoles along z, the contiguous axis), Udd(0) = 0
    and the 1/N normalisation."""
    gold = read_golden("survey_p4_plane_wave.txt")
    shape, d = (12, 8, 6), (0.3, 0.5, 0.7)
    o = make(oracle, shape, d)
    L = [s * dd for s, dd in zip(shape, d)]
    x, y, z = [inputs.coords(s, dd) for s, dd in zip(shape, d)]
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    amp = 0.37
    cases = [((0, 0, 1), gold["parallel_z"]), ((0, 0, 2), gold["parallel_z"]),
             ((1, 0, 0), gold["perpendicular_z"]), ((0, 3, 0), gold["perpendicular_z"]),
             ((2, 1, 1), None), ((-1, 2, -2), None)]
    for m, udd_expected in cases:
        q = [2 * np.pi * mi / Li for mi, Li in zip(m, L)]
        udd = (4 * np.pi / 3) * (3 * q[2] ** 2 / (q[0] ** 2 + q[1] ** 2 + q[2] ** 2) - 1)
        if udd_expected is not None:
            assert abs(udd - udd_expected) < 1e-11
        wave = np.cos(q[0] * X + q[1] * Y + q[2] * Z + 0.4)
        phi = o.dipolar(np.ascontiguousarray(1.0 + amp * wave))
        assert np.max(np.abs(phi - udd * amp * wave)) <= 2e-14 * abs(udd) + 1e-14, m


def test_p5_isotropic_gaussian_cubic_symmetry(oracle):
    """Isotropic density on a cubic grid: sum Phi n = 0 (cubic symmetry kills sum (3kz^2/k^2-1)|n_k|^2)."""
    shape, d = (16, 16, 16), (0.5, 0.5, 0.5)
    o = make(oracle, shape, d)
    x = inputs.coords(16, 0.5)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    n = np.exp(-(X * X + Y * Y + Z * Z))
    phi = o.dipolar(np.ascontiguousarray(n))
    assert abs(np.sum(phi * n)) <= 1e-13 * np.sum(n * n)


def f_kappa(k):
    if abs(k - 1.0) < 1e-12:
        return 0.0
    if k < 1:
        s = math.sqrt(1 - k * k)
        return (1 + 2 * k * k) / (1 - k * k) - 3 * k * k * math.atanh(s) / s ** 3
    s = math.sqrt(k * k - 1)
    return (1 + 2 * k * k) / (1 - k * k) + 3 * k * k * math.atan(s) / s ** 3


def test_p6_gaussian_dipolar_energy_closed_form(oracle):
    """Gaussian density exp(-rho^2/s_rho^2 - z^2/s_z^2): int Phi n = -(4 pi/3) f(kappa) int n^2,
    kappa = s_rho/s_z (standard dipolar anisotropy function; f(sqrt 2) = -5 + 3 pi/2).
    Periodic images limit the accuracy to O((sigma/L)^3)."""
    assert abs(f_kappa(math.sqrt(2.0)) - (-5 + 1.5 * math.pi)) < 1e-12
    shape, d = (48, 48, 48), (0.5, 0.5, 0.5)
    o = make(oracle, shape, d)
    x = inputs.coords(48, 0.5)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    for s_rho, s_z in [(1.0, 2.0), (2.0, 1.0), (1.5, 1.0)]:
        n = np.exp(-(X * X + Y * Y) / s_rho ** 2 - Z * Z / s_z ** 2)
        phi = o.dipolar(np.ascontiguousarray(n))
        got = np.sum(phi * n) / np.sum(n * n)
        want = -(4 * np.pi / 3) * f_kappa(s_rho / s_z)
        assert abs(got - want) <= 5e-3 * abs(want) + 2e-3, (s_rho, s_z, got, want)


def test_p6b_dipolar_vs_numpy_fft_random_density(oracle):
    """Random density on an unequal grid against numpy.fft (a library the oracle does not use)."""
    shape, d = (6, 9, 8), (0.4, 0.3, 0.6)
    o = make(oracle, shape, d)
    rng = np.random.default_rng(11)
    n = rng.random(shape)
    k = [2 * np.pi * np.fft.fftfreq(s, dd) for s, dd in zip(shape, d)]
    KX, KY, KZ = np.meshgrid(*k, indexing="ij")
    k2 = KX ** 2 + KY ** 2 + KZ ** 2
    k2[0, 0, 0] = 1.0
    U = (4 * np.pi / 3) * (3 * KZ ** 2 / k2 - 1)
    U[0, 0, 0] = 0.0
    ref = np.fft.ifftn(U * np.fft.fftn(n)).real
    assert np.max(np.abs(o.dipolar(n) - ref)) <= 1e-13 * np.max(np.abs(ref))


# ------------------------------------------------------------------------------------------
# P7: Crank-Nicolson line solve = dense Gaussian elimination (BJ:north_star check 2)
# ------------------------------------------------------------------------------------------

def dense_cn(line, r):
    """psi' on the interior nodes 1..n-2 by dense solve; end nodes are the Dirichlet boundary."""
    n = line.size
    m = n - 2
    A = np.zeros((m, m), dtype=np.complex128)
    B = np.zeros((m, m), dtype=np.complex128)
    for j in range(m):
        A[j, j], B[j, j] = 1 + 2 * r, 1 - 2 * r
        if j:
            A[j, j - 1] = A[j - 1, j] = -r
            B[j, j - 1] = B[j - 1, j] = r
    out = np.zeros(n, dtype=np.complex128)
    out[1:-1] = np.linalg.solve(A, B @ line[1:-1])
    return out


@pytest.mark.parametrize("mode", [IMAG, REAL])
@pytest.mark.parametrize("shape", [(5, 6, 7), (12, 9, 4), (4, 4, 4)])
def test_p7_sweep_is_dense_solve(oracle, mode, shape):
    d = (0.5, 0.25, 0.1)
    for dt in (0.005, 0.5):                           # r from 0.005 to 12.5 (times i in real time)
        o = make(oracle, shape, d, dt=dt, mode=mode)
        for axis in range(3):
            psi = rand_c(shape, 100 + axis)           # non-zero faces: must be treated as 0
            ref = np.empty_like(psi)
            rr = dt / (4 * d[axis] ** 2)
            r = rr if mode == IMAG else 1j * rr
            moved = np.moveaxis(psi, axis, -1)
            refm = np.moveaxis(ref, axis, -1)
            for idx in np.ndindex(moved.shape[:-1]):
                refm[idx] = dense_cn(moved[idx], r)
            got = psi.copy()
            assert o.sweep(got, axis) == 0
            assert np.max(np.abs(got - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))


# ------------------------------------------------------------------------------------------
# nonlinear / potential factor
# ------------------------------------------------------------------------------------------

@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_nonlinear_trap_only_closed_form(oracle, mode):
    """g = gdd = 0: psi <- exp(-dt V) psi or exp(-i dt V) psi with V = (g^2x^2 + n^2y^2 + l^2z^2)/2,
    gamma <-> x (slowest axis), nu <-> y, lambda <-> z (contiguous)."""
    shape, d, dt, trap = (6, 8, 10), (0.3, 0.4, 0.5), 0.02, (1.3, 0.7, 2.1)
    o = make(oracle, shape, d, dt=dt, trap=trap, g=0.0, gdd=0.0, mode=mode)
    psi = rand_c(shape, 5)
    x, y, z = [inputs.coords(s, dd) for s, dd in zip(shape, d)]
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    V = 0.5 * (trap[0] ** 2 * X ** 2 + trap[1] ** 2 * Y ** 2 + trap[2] ** 2 * Z ** 2)
    ref = psi * (np.exp(-dt * V) if mode == IMAG else np.exp(-1j * dt * V))
    got = psi.copy()
    assert o.nonlinear(got) == 0
    assert np.max(np.abs(got - ref)) <= 1e-14 * np.max(np.abs(ref))


@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_nonlinear_contact_and_dipolar_vs_numpy(oracle, mode):
    shape, d, dt, trap, g, gdd = (6, 4, 8), (0.3, 0.4, 0.5), 0.02, (1.0, 0.5, 2.0), 3.0, 1.7
    o = make(oracle, shape, d, dt=dt, trap=trap, g=g, gdd=gdd, mode=mode)
    psi = 0.6 * rand_c(shape, 6)
    n = np.abs(psi) ** 2
    phi = brute_dft3(brute_dipolar_kernel(shape, d) * brute_dft3(n, -1), +1).real / n.size
    x, y, z = [inputs.coords(s, dd) for s, dd in zip(shape, d)]
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    H = 0.5 * (trap[0] ** 2 * X ** 2 + trap[1] ** 2 * Y ** 2 + trap[2] ** 2 * Z ** 2) + g * n + gdd * phi
    ref = psi * (np.exp(-dt * H) if mode == IMAG else np.exp(-1j * dt * H))
    got = psi.copy()
    assert o.nonlinear(got) == 0
    assert np.max(np.abs(got - ref)) <= 1e-13


def brute_dipolar_kernel(shape, d):
    ks = []
    for s, dd in zip(shape, d):
        m = np.arange(s)
        f = np.where(m <= s // 2, m, m - s)
        ks.append(2 * np.pi * f / (s * dd))
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    k2 = KX ** 2 + KY ** 2 + KZ ** 2
    k2[0, 0, 0] = 1.0
    U = (4 * np.pi / 3) * (3 * KZ ** 2 / k2 - 1)
    U[0, 0, 0] = 0.0
    return U


# ------------------------------------------------------------------------------------------
# whole step on a tiny grid against a dense-matrix restatement (different algorithms for every
# sub-result: O(n^2) DFT instead of the FFT, dense solve instead of Thomas)
# ------------------------------------------------------------------------------------------

def dense_step(psi, shape, d, dt, trap, g, gdd, mode):
    n = np.abs(psi) ** 2
    phi = brute_dft3(brute_dipolar_kernel(shape, d) * brute_dft3(n, -1), +1).real / n.size
    x, y, z = [inputs.coords(s, dd) for s, dd in zip(shape, d)]
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    H = 0.5 * (trap[0] ** 2 * X ** 2 + trap[1] ** 2 * Y ** 2 + trap[2] ** 2 * Z ** 2) + g * n + gdd * phi
    psi = psi * (np.exp(-dt * H) if mode == IMAG else np.exp(-1j * dt * H))
    for axis in range(3):
        rr = dt / (4 * d[axis] ** 2)
        r = rr if mode == IMAG else 1j * rr
        moved = np.moveaxis(psi, axis, -1).copy()
        for idx in np.ndindex(moved.shape[:-1]):
            moved[idx] = dense_cn(moved[idx], r)
        psi = np.moveaxis(moved, -1, axis)
    if mode == IMAG:
        psi = psi / np.sqrt(np.sum(np.abs(psi) ** 2) * d[0] * d[1] * d[2])
    return np.ascontiguousarray(psi)


@pytest.mark.parametrize("mode", [IMAG, REAL])
def test_step_vs_dense_restatement(oracle, mode):
    shape, d, dt, trap, g, gdd = (6, 8, 10), (0.5, 0.4, 0.3), 0.01, (1.0, 0.8, 1.5), 4.0, 2.5
    o = make(oracle, shape, d, dt=dt, trap=trap, g=g, gdd=gdd, mode=mode)
    psi = inputs.random_state(shape, 3) * 0.5
    ref = psi.copy()
    for _ in range(5):
        ref = dense_step(ref, shape, d, dt, trap, g, gdd, mode)
    got = psi.copy()
    assert o.step(got, 5) == 0
    assert np.max(np.abs(got - ref)) <= 1e-13
    for face in (got[0], got[-1], got[:, 0], got[:, -1], got[:, :, 0], got[:, :, -1]):
        assert np.all(face == 0)                      # Dirichlet faces are exactly 0 after a step


# ------------------------------------------------------------------------------------------
# P8: real-time norm conservation (BJ:north_star check 4)
# ------------------------------------------------------------------------------------------

def test_p8_real_time_norm_conservation(oracle):
    cfg = inputs.scaled(replace(inputs.CONFIGS["C1"], mode=REAL), (32, 32, 32))
    cfg = replace(cfg, d=(0.5, 0.5, 0.5))
    o = oracle.Oracle(*cfg.create_args())
    psi = inputs.initial_state(cfg)
    n0 = o.norm(psi)
    assert abs(n0 - 1) <= 1e-14
    for _ in range(50):
        assert o.step(psi, 1) == 0
        assert abs(o.norm(psi) - n0) <= 1e-12


# ------------------------------------------------------------------------------------------
# R#5: in imaginary time a real psi stays real, and the real and imaginary parts never mix
# (every factor of the step is real).  This is what lets the library carry psi as plain doubles
# (DGPE_IMAG_RPSI) and still be compared with this complex oracle.
# ------------------------------------------------------------------------------------------

def test_imaginary_time_keeps_a_real_psi_exactly_real(oracle):
    cfg = inputs.scaled(inputs.CONFIGS["C1"], (16, 12, 20))
    o = oracle.Oracle(*cfg.create_args())
    psi = inputs.random_state(cfg.shape, 17)
    re = np.ascontiguousarray(psi.real.astype(np.complex128))
    for stage in (lambda a: o.nonlinear(a), lambda a: o.sweep(a, 0), lambda a: o.sweep(a, 1), lambda a: o.sweep(a, 2)):
        a = re.copy()
        stage(a)
        assert np.all(a.imag == 0)
    a = re.copy()
    assert o.step(a, 5) == 0
    assert np.all(a.imag == 0)
    # the sweeps are real-linear: the sweep of the real part is the real part of the sweep
    for axis in range(3):
        full, part = psi.copy(), re.copy()
        o.sweep(full, axis)
        o.sweep(part, axis)
        assert np.array_equal(full.real, part.real)


# ------------------------------------------------------------------------------------------
# P9: observables on a Gaussian (closed forms; spectrally accurate on these grids)
# ------------------------------------------------------------------------------------------

def test_p9_gaussian_observables_closed_forms(oracle):
    gold = read_golden("survey_p13_c1_noisefree.txt")
    cfg = replace(inputs.CONFIGS["C1"], noise=0.0)
    o = oracle.Oracle(*cfg.create_args())
    psi = inputs.initial_state(cfg)
    w, d = 1.0, 0.25
    T = 3 * (1 - math.exp(-w * d * d / 4)) / (d * d)       # link-sum kinetic term of a sampled Gaussian
    V = 3 * w / 4
    gn = cfg.g * (w / (2 * math.pi)) ** 1.5
    terms = o.energy_terms(psi)
    assert abs(terms[0] - T) <= 1e-11 and abs(T - gold[(0, "T")]) <= 1e-11
    assert abs(terms[1] - V) <= 1e-11 and abs(V - gold[(0, "V")]) <= 1e-11
    assert abs(terms[2] - gn) <= 1e-11 and abs(gn - gold[(0, "gn")]) <= 1e-11
    assert abs(terms[3]) <= 1e-12                          # P5: isotropic => dipolar term vanishes
    assert abs(o.chempot(psi) - gold[(0, "mu")]) <= 1e-11
    assert abs(o.energy(psi) - gold[(0, "energy")]) <= 1e-11
    rms = o.rms(psi)
    for a in range(3):
        assert abs(rms[a] - math.sqrt(0.5)) <= 1e-11
    assert abs(rms[3] - math.sqrt(1.5)) <= 1e-11
    assert abs(o.norm(psi) - 1.0) <= 1e-13


def test_p9_anisotropic_gaussian_rms_and_potential(oracle):
    """<x_a^2> = 1/(2 w_a), <V> = sum Omega_a^2/(4 w_a), T = sum (1-exp(-w_a d_a^2/4))/d_a^2."""
    shape, d = (48, 40, 64), (0.3, 0.35, 0.2)
    wg, trap = (1.2, 0.9, 2.0), (0.7, 1.1, 1.9)
    cfg = inputs.Config("t", shape, d, 0.01, trap, 0.0, 0.0, IMAG, 1, 9, wg, noise=0.0)
    o = oracle.Oracle(*cfg.create_args())
    psi = inputs.initial_state(cfg) * 1.7                  # observables divide by the norm
    rms = o.rms(psi)
    for a in range(3):
        assert abs(rms[a] - math.sqrt(1 / (2 * wg[a]))) <= 1e-9
    t = o.energy_terms(psi)
    assert abs(t[1] - sum(trap[a] ** 2 / (4 * wg[a]) for a in range(3))) <= 1e-9
    assert abs(t[0] - sum((1 - math.exp(-wg[a] * d[a] ** 2 / 4)) / d[a] ** 2 for a in range(3))) <= 1e-9
    assert abs(o.norm(psi) - 1.7 ** 2) <= 1e-12


# ------------------------------------------------------------------------------------------
# P10-P12: g = gdd = 0 imaginary-time limit (BJ:north_star check 3).  The step map is linear and
# separable, so its fixed point is the outer product of the dominant eigenvectors of the 1-D maps
# M_a = A_a^{-1} B_a diag(exp(-dt V_a)), obtained here by dense linear algebra.
# ------------------------------------------------------------------------------------------

def one_d_map(n, d, dt, omega):
    m = n - 2
    r = dt / (4 * d * d)
    A = np.diag(np.full(m, 1 + 2 * r)) + np.diag(np.full(m - 1, -r), 1) + np.diag(np.full(m - 1, -r), -1)
    B = np.diag(np.full(m, 1 - 2 * r)) + np.diag(np.full(m - 1, r), 1) + np.diag(np.full(m - 1, r), -1)
    x = inputs.coords(n, d)[1:-1]
    return np.linalg.solve(A, B) @ np.diag(np.exp(-dt * 0.5 * omega ** 2 * x ** 2)), x


def test_p10_p12_harmonic_ground_state(oracle):
    shape, d, dt, trap = (32, 32, 32), (0.5, 0.5, 0.5), 0.02, (1.0, 1.0, 1.0)
    cfg = inputs.Config("t", shape, d, dt, trap, 0.0, 0.0, IMAG, 1, 12, (1.0, 1.0, 1.0), noise=1e-3)
    o = oracle.Oracle(*cfg.create_args())
    psi = inputs.initial_state(cfg)
    assert o.step(psi, 1500) == 0
    # dense 1-D fixed point
    M, x = one_d_map(32, 0.5, dt, 1.0)
    ev, vec = np.linalg.eig(M)
    k = np.argmax(ev.real)
    v = np.real(vec[:, k])
    v = v / np.sqrt(np.sum(v * v) * 0.5) * np.sign(v[len(v) // 2])
    full = np.zeros(32)
    full[1:-1] = v
    ref = np.einsum("i,j,k->ijk", full, full, full)
    assert np.max(np.abs(psi - ref)) <= 1e-10                          # fixed point of the step
    # P12: the decay rate before renormalising is the dominant eigenvalue cubed
    one = psi.copy()
    o.nonlinear(one)
    for a in range(3):
        o.sweep(one, a)
    assert abs(o.norm(one) - ev.real[k] ** 6) <= 1e-12
    # P10: mu against the lowest eigenvalue of the discrete 1-D Hamiltonian and the continuum value
    m = 30
    Hm = (np.diag(np.full(m, 1.0 / 0.25)) + np.diag(np.full(m - 1, -0.5 / 0.25), 1) +
          np.diag(np.full(m - 1, -0.5 / 0.25), -1) + np.diag(0.5 * x * x))
    e0 = np.linalg.eigvalsh(Hm)[0]
    mu = o.chempot(psi)
    assert abs(mu - 3 * e0) <= 5e-4                 # Lie-splitting offset O(dt^2)
    assert abs(mu - 1.5) <= 3 * (0.5 ** 2) / 32 + 2e-3   # (gamma+nu+lambda)/2 up to O(dx^2)
    # mu of the dense fixed point by the same Rayleigh quotient, computed independently
    t1 = 0.5 * np.sum(np.diff(np.concatenate([[0.0], full, [0.0]])) ** 2) / 0.25 / np.sum(full ** 2)
    v1 = np.sum(0.5 * inputs.coords(32, 0.5) ** 2 * full ** 2) / np.sum(full ** 2)
    assert abs(mu - 3 * (t1 + v1)) <= 1e-10
    # P11: rms
    rms = o.rms(psi)
    assert abs(rms[0] - math.sqrt(0.5)) <= 2e-2


# ------------------------------------------------------------------------------------------
# P13: whole imaginary-time step with interactions against the survey's independent values
# ------------------------------------------------------------------------------------------

def test_p13_c1_noisefree_third_implementation(oracle):
    gold = read_golden("survey_p13_c1_noisefree.txt")
    cfg = replace(inputs.CONFIGS["C1"], noise=0.0)
    o = oracle.Oracle(*cfg.create_args())
    psi = inputs.initial_state(cfg)
    done = 0
    for step in (1, 10, 100):
        assert o.step(psi, step - done) == 0
        done = step
        vals = {"mu": o.chempot(psi), "energy": o.energy(psi)}
        rms = o.rms(psi)
        vals.update(rms_x=rms[0], rms_y=rms[1], rms_z=rms[2], rms_r=rms[3],
                    psi_centre=abs(psi[32, 32, 32]))
        for (s, name), want in gold.items():
            if s == step:
                assert abs(vals[name] - want) <= 2e-11 * max(1.0, abs(want)), (step, name, vals[name], want)
        assert abs(rms[0] - rms[1]) <= 1e-13
        assert abs(o.norm(psi) - 1.0) <= 1e-13
        assert np.max(np.abs(psi.imag)) == 0.0       # real input stays real in imaginary time


def test_p13_c2_noisefree_first_step(oracle):
    gold = read_golden("survey_p13_c2_noisefree.txt")
    cfg = replace(inputs.CONFIGS["C2"], noise=0.0)
    o = oracle.Oracle(*cfg.create_args())
    psi = inputs.initial_state(cfg)
    assert abs(o.chempot(psi) - gold[(0, "mu")]) <= 2e-11 * gold[(0, "mu")]
    assert abs(o.energy(psi) - gold[(0, "energy")]) <= 2e-11 * gold[(0, "energy")]
    assert o.step(psi, 1) == 0
    assert abs(o.chempot(psi) - gold[(1, "mu")]) <= 2e-11 * gold[(1, "mu")]
    assert abs(o.energy(psi) - gold[(1, "energy")]) <= 2e-11 * gold[(1, "energy")]


# ------------------------------------------------------------------------------------------
# argument checking
# ------------------------------------------------------------------------------------------

def test_nonfinite_norm_status_and_no_clamp(oracle):
    """R#18 / SURVEY 8(b): the imaginary-time renormalisation has no clamp.  A zero state has norm 0 (psi / sqrt(0)), an
    overflowing exponential gives inf: both must come back as ODGPE_ERR_NONFINITE, the status the CUDA path is compared
    with for the literal 200-step C4 call; a healthy state returns OK, and real time never reports it (no norm taken)."""
    shape = (8, 8, 8)
    phys = (0.5, 0.5, 0.5, 0.01, 1.0, 1.0, 1.0, 1.0, 1.0)
    Oi, Or = oracle.Oracle(*shape, *phys, 0), oracle.Oracle(*shape, *phys, 1)
    good = inputs.random_state(shape, 61) * 0.3
    assert Oi.step(good.copy(), 2) == oracle.OK
    zero = np.zeros(shape, dtype=np.complex128)
    assert Oi.step(zero, 1) == oracle.ERR_NONFINITE                   # norm = 0
    assert Or.step(np.zeros(shape, dtype=np.complex128), 1) == oracle.OK
    # exp(-dt H) with H = g |psi|^2 hugely negative (attractive contact term): overflow -> inf norm
    Oneg = oracle.Oracle(*shape, 0.5, 0.5, 0.5, 0.01, 1.0, 1.0, 1.0, -1.0e6, 0.0, 0)
    big = inputs.random_state(shape, 62) * 30.0
    a = big.copy()
    assert Oneg.step(a, 1) == oracle.ERR_NONFINITE
    assert not np.all(np.isfinite(a.view(np.float64)))                # nothing was clamped
    # the status is sticky within a call: a later finite norm does not clear it
    b = zero.copy()
    assert Oi.step(b, 3) == oracle.ERR_NONFINITE


def test_create_rejects_bad_arguments(oracle):
    good = list(inputs.CONFIGS["C1"].create_args())
    for pos, bad in [(0, 3), (3, 0.0), (4, -1.0), (6, 0.0), (12, 2)]:
        args = list(good)
        args[pos] = bad
        with pytest.raises(ValueError):
            oracle.Oracle(*args)


# ------------------------------------------------------------------------------------------
# input recipe: what `bench.py --rpsi` and tests/test_gpu_rpsi.py rely on
# ------------------------------------------------------------------------------------------

def test_imaginary_time_initial_states_are_real_normalised_and_zero_faced():
    for name, shape in (("C1", (64, 64, 64)), ("C2", (32, 48, 64)), ("C4", (48, 32, 64))):
        cfg = inputs.CONFIGS[name] if inputs.CONFIGS[name].shape == shape else inputs.scaled(inputs.CONFIGS[name], shape)
        psi = inputs.initial_state(cfg)
        assert psi.dtype == np.complex128 and psi.shape == shape
        assert np.all(psi.imag == 0)                      # Gaussian x (1 + noise): real, so the real-valued path takes it as is
        assert abs(np.sum(np.abs(psi) ** 2) * cfg.d[0] * cfg.d[1] * cfg.d[2] - 1) <= 1e-13
        for face in (psi[0], psi[-1], psi[:, 0], psi[:, -1], psi[:, :, 0], psi[:, :, -1]):
            assert np.all(face == 0)
    c5 = inputs.initial_state(inputs.scaled(inputs.CONFIGS["C5"], (24, 24, 12)))
    assert np.any(c5.imag != 0)                           # the seeded phase field makes C5 genuinely complex
