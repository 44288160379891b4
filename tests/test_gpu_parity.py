"""GPU parity tests proper (-m gpu): the CUDA path, called through the C-ABI (ctypes binding), against
the CPU oracle on the same seeded inputs, element by element; and at BASELINE.json's full sizes via
sampled lines the oracle solves one by one and closed forms that hold at any size.

Tolerances (BJ:north_star): max|psi_gpu - psi_ref| <= 1e-12 after one step, <= 1e-10 after 100 steps;
mu and E to 1e-10 relative.  Parity windows follow DESIGN.md section 4 (collapse regime, R#27)."""
import numpy as np
import pytest
import torch

from paper_1610_05329_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12
TOL_100 = 1e-10
TOL_OBS = 1e-10


@pytest.fixture(scope="module")
def gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1610_05329_b200 import binding
    binding.lib()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def pair(gpu, oracle, shape, d, dt, trap, g, gdd, mode):
    return (gpu.Dgpe(*shape, *d, dt, *trap, g, gdd, mode), oracle.Oracle(*shape, *d, dt, *trap, g, gdd, mode))


# shapes span: one tile, ragged last tiles (line counts not multiples of 8), radix 3, several FFT passes,
# nz = 2*odd, minimum size 4, non-cubic
# (the last three: the 768- and 384-point kernels of BJ:configs[4] -- TMA-fed sweeps with 96 chunks per line,
# four-pass FFTs with a radix-3 pass, the 384-point z-line kernels -- on thin boxes the oracle finishes fast)
STAGE_SHAPES = [(4, 4, 4), (8, 8, 8), (6, 9, 12), (12, 18, 16), (27, 32, 6), (16, 24, 36), (64, 64, 64),
                (48, 96, 128), (9, 4, 18), (768, 8, 64), (16, 768, 128), (8, 384, 384),
                # radix 5 and 7 (SV section 8f NEXT-1): generic plans, and the specialised 160/240/480/500
                # lengths of the paper's own grids (480^3, 480x480x500, 480x480x250: P:L75, L96, L111)
                (10, 14, 20), (35, 25, 50), (7, 5, 98), (480, 8, 70), (8, 500, 250), (16, 240, 160), (8, 160, 320),
                (8, 8, 480), (12, 8, 500), (8, 8, 640), (8, 12, 240),
                # lengths whose largest radix is small (more than 128 butterflies per pass: several per thread)
                (486, 4, 6), (4, 729, 4), (4, 6, 972), (686, 4, 10), (4, 6, 600)]


@pytest.mark.parametrize("shape", STAGE_SHAPES)
@pytest.mark.parametrize("mode", [0, 1])
def test_stage_parity(gpu, oracle, shape, mode):
    G, O = pair(gpu, oracle, shape, (0.3, 0.25, 0.2), 0.01, (1.0, 0.7, 1.3), 5.0, 3.0, mode)
    psi = inputs.random_state(shape, 3) * 0.3
    # (a) dipolar mean field
    phi = G.dipolar(dev(psi)).cpu().numpy()
    ref = O.dipolar(np.ascontiguousarray(psi.real ** 2 + psi.imag ** 2))
    assert np.max(np.abs(phi - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    # (a)+(b) nonlinear exponential
    t, a = dev(psi), psi.copy()
    G.nonlinear(t)
    O.nonlinear(a)
    assert np.max(np.abs(t.cpu().numpy() - a)) <= TOL_1
    # (c) each sweep
    for axis in range(3):
        t, a = dev(psi), psi.copy()
        G.sweep(t, axis)
        O.sweep(a, axis)
        out = t.cpu().numpy()
        assert np.max(np.abs(out - a)) <= TOL_1, axis
        # Dirichlet end nodes are written as exact zeros
        sl = [slice(None)] * 3
        for end in (0, -1):
            sl[axis] = end
            assert np.all(out[tuple(sl)] == 0)
    # observables
    t = dev(psi)
    got = [G.norm(t), *G.rms(t), *G.energy_terms(t), G.chempot(t), G.energy(t)]
    exp = [O.norm(psi), *O.rms(psi), *O.energy_terms(psi), O.chempot(psi), O.energy(psi)]
    for x, y in zip(got, exp):
        assert abs(x - y) <= TOL_OBS * max(1.0, abs(y))


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("dt", [0.5, 5.0, 40.0])
def test_sweeps_with_large_r_need_the_long_lookback(gpu, oracle, mode, dt):
    """r = dt/(4 d^2) up to 250: the chunk factors are O(1), so the inflow look-back spans many chunks."""
    # (64, 48, 96): generic z kernel; (8, 384, 128): the TMA-fed y sweep and the warp-per-line z sweep, both
    # reading the global tables because the elimination factors do not converge within a chunk
    for shape in [(64, 48, 96), (8, 384, 128)]:
        G, O = pair(gpu, oracle, shape, (0.3, 0.25, 0.2), dt, (1.0, 1.0, 1.0), 0.0, 0.0, mode)
        psi = inputs.random_state(shape, 5)
        for axis in range(3):
            t, a = dev(psi), psi.copy()
            G.sweep(t, axis)
            O.sweep(a, axis)
            assert np.max(np.abs(t.cpu().numpy() - a)) <= 1e-12 * (1 + dt), (shape, axis)


def _smooth_lengths(lo=4, hi=1024):
    out = []
    for n in range(lo, hi + 1):
        m = n
        for f in (2, 3, 5, 7, 11, 13):
            while m % f == 0:
                m //= f
        if m == 1:
            out.append(n)
    return out


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_every_supported_length_on_every_axis(gpu, oracle, axis, mode):
    """One full step (imaginary or real time) for EVERY length 2^a 3^b 5^c 7^d 11^e 13^f in [4, 1024] on each axis (thin box in
    the other two), against the oracle: every plan, specialised or generic, launches and is right."""
    worst = 0.0
    for n in _smooth_lengths():
        if axis == 2 and n % 2:
            continue
        shape = [8, 8, 8]
        shape[axis] = n
        shape = tuple(shape)
        G, O = pair(gpu, oracle, shape, (0.3, 0.25, 0.2), 0.01, (1.0, 0.7, 1.3), 5.0, 3.0, mode)
        psi = inputs.random_state(shape, 100 + n) * 0.3
        t, a = dev(psi), psi.copy()
        assert G.step(t, 1) == O.step(a, 1) == 0, shape
        err = float(np.max(np.abs(t.cpu().numpy() - a)))
        assert err <= TOL_1, (shape, err)
        worst = max(worst, err)
        G.close()
    print(f"mode {mode} axis {axis}: worst |dpsi| over all lengths = {worst:.2e}")


def run_both(gpu, oracle, cfg, checkpoints, psi0=None):
    """Step GPU and oracle side by side; at each checkpoint return (step, max|dpsi|, obs_gpu, obs_ref)."""
    psi0 = inputs.initial_state(cfg) if psi0 is None else psi0
    G, O = gpu.Dgpe(*cfg.create_args()), oracle.Oracle(*cfg.create_args())
    t, a = dev(psi0), psi0.copy()
    done, out = 0, []
    for cp in checkpoints:
        rc_g = G.step(t, cp - done)
        rc_o = O.step(a, cp - done)
        done = cp
        assert rc_g == rc_o
        err = float(np.max(np.abs(t.cpu().numpy() - a)))
        og = [G.norm(t), G.chempot(t), G.energy(t), *G.rms(t)]
        orf = [O.norm(a), O.chempot(a), O.energy(a), *O.rms(a)]
        out.append((cp, err, og, orf))
    return out, t, a


def check_obs(og, orf):
    for x, y in zip(og, orf):
        assert abs(x - y) <= TOL_OBS * max(1.0, abs(y)), (og, orf)


def test_c1_full_config_1_and_100_steps(gpu, oracle):
    """BJ:configs[0], literally: 64^3 imaginary time, 100 steps with renormalisation each step."""
    res, t, a = run_both(gpu, oracle, inputs.CONFIGS["C1"], [1, 10, 100])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100), (cp, err)
        check_obs(og, orf)
        assert abs(og[0] - 1.0) <= 1e-13          # imaginary time returns unit norm


def test_c2_128cubed_1_and_20_steps(gpu, oracle):
    """BJ:configs[1] on its full 128^3 grid (smooth window)."""
    res, _, _ = run_both(gpu, oracle, inputs.CONFIGS["C2"], [1, 20])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100), (cp, err)
        check_obs(og, orf)


def test_c3_protocol_scaled_relax_then_quench_real_time(gpu, oracle):
    """BJ:configs[2] protocol on a 48^3 box with the same spacings: imaginary-time relaxation with
    g = 80, then real time after the quench to g = 64; norm conserved at every checkpoint."""
    cfg = inputs.scaled(inputs.CONFIGS["C3"], (48, 48, 48))
    res, t, a = run_both(gpu, oracle, cfg.relax, [1, 60])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100)
        check_obs(og, orf)
    # quench: continue each side from ITS OWN relaxed state (they agree to TOL_100)
    G, O = gpu.Dgpe(*cfg.create_args()), oracle.Oracle(*cfg.create_args())
    n0 = G.norm(t)
    done = 0
    for cp in (1, 10, 100):
        G.step(t, cp - done)
        O.step(a, cp - done)
        done = cp
        assert np.max(np.abs(t.cpu().numpy() - a)) <= 2 * TOL_100
        assert abs(G.norm(t) - n0) <= 1e-12        # BJ:north_star check (4)
        check_obs([G.chempot(t), G.energy(t), *G.rms(t)], [O.chempot(a), O.energy(a), *O.rms(a)])


def test_c5_scaled_non_cubic_radix3_real_time(gpu, oracle):
    """BJ:configs[4] on 96x96x48 (same spacings, radix-3 passes on every axis): seeded phase field,
    real time, norm and energy tracked."""
    cfg = inputs.scaled(inputs.CONFIGS["C5"], (96, 96, 48))
    res, _, _ = run_both(gpu, oracle, cfg, [1, 10, 100])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100), (cp, err)
        check_obs(og, orf)
        assert abs(og[0] - 1.0) <= 1e-12


def test_c4_physics_scaled_smooth_window_and_nonfinite_status(gpu, oracle):
    """BJ:configs[3] physics on a 64^3 box: parity inside the smooth window (steps 1, 10), and both
    sides must agree on the status of the literal long call (collapse regime, R#27: no clamp)."""
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (64, 64, 64))
    res, t, a = run_both(gpu, oracle, cfg, [1, 10])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100), (cp, err)
        check_obs(og, orf)
    G, O = gpu.Dgpe(*cfg.create_args()), oracle.Oracle(*cfg.create_args())
    rc_g, rc_o = G.step(t, 190), O.step(a, 190)
    assert rc_g == rc_o
    if rc_g == gpu.ERR_NONFINITE:
        assert "norm" in gpu.last_error()


def test_256cubed_single_real_time_step(gpu, oracle):
    """BJ:configs[2] grid at full size (256^3, real-time handle), one step from the seeded Gaussian."""
    cfg = inputs.CONFIGS["C3"]
    psi0 = inputs.initial_state(cfg)
    G, O = gpu.Dgpe(*cfg.create_args()), oracle.Oracle(*cfg.create_args())
    t, a = dev(psi0), psi0.copy()
    G.step(t, 1)
    O.step(a, 1)
    assert np.max(np.abs(t.cpu().numpy() - a)) <= TOL_1
    assert abs(G.norm(t) - 1.0) <= 1e-12


def test_edge_cases(gpu, oracle):
    G, O = pair(gpu, oracle, (8, 12, 4), (0.5, 0.4, 0.3), 0.01, (1.0, 1.0, 1.0), 1.0, 1.0, 0)
    psi = inputs.random_state((8, 12, 4), 9)
    t = dev(psi)
    before = t.clone()
    assert G.step(t, 0) == gpu.OK                   # empty call: no-op
    assert torch.equal(t, before)
    z = torch.zeros((8, 12, 4), dtype=torch.complex128, device="cuda")
    assert G.step(z, 1) == gpu.ERR_NONFINITE        # zero state: norm 0 -> same status as the oracle
    a = np.zeros((8, 12, 4), dtype=np.complex128)
    assert O.step(a, 1) == oracle.ERR_NONFINITE
    with pytest.raises(TypeError):
        G.step(t.to(torch.complex64), 1)
    with pytest.raises(gpu.DgpeError):
        G.sweep(t, 3)
    # un-normalised, non-zero faces on input: the step ignores the faces in the sweeps (R#8)
    psi2 = inputs.random_state((8, 12, 4), 10, zero_faces=False) * 3.0
    t, a = dev(psi2), psi2.copy()
    assert G.step(t, 2) == O.step(a, 2) == 0
    assert np.max(np.abs(t.cpu().numpy() - a)) <= TOL_1


def test_step_host_matches_device_path(gpu):
    cfg = inputs.CONFIGS["C1"]
    psi0 = inputs.initial_state(cfg)
    G = gpu.Dgpe(*cfg.create_args())
    t = dev(psi0)
    G.step(t, 3)
    hp = torch.from_numpy(psi0.copy()).pin_memory()
    assert G.step_host(hp, 3) == gpu.OK
    assert torch.equal(hp, t.cpu())                 # same kernels, deterministic reductions: bit-identical


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("opt", [{"generic": 1}, {"tma": 0}, {"tma": 2}, {"graph": 0}, {"prefetch": 0}, {"tma_fft": 0}])
def test_kernel_variants_agree(gpu, mode, opt):
    """The library carries two kernel sets (specialised and generic) and dgpe_create_ex options
    for A/B runs; every variant must give the same step to rounding (different summation orders only)."""
    shape = (64, 384, 128)
    args = (*shape, 0.3, 0.25, 0.2, 0.004, 1.0, 0.7, 1.3, 5.0, 3.0, mode)
    psi = inputs.random_state(shape, 21) * 0.05
    ref = dev(psi)
    gpu.Dgpe(*args).step(ref, 3)
    alt = dev(psi)
    gpu.Dgpe(*args, options=opt).step(alt, 3)
    assert float((alt - ref).abs().max()) <= 1e-13


@pytest.mark.parametrize("shape", [(8, 8, 64), (8, 6, 384), (8, 8, 100)])
@pytest.mark.parametrize("theta_max", [20.0, 3.0e4, 5.0e9])
def test_real_time_phase_range_of_the_fast_sincos(gpu, oracle, shape, theta_max):
    """Real time: exp(-i dt H) through the branch-free sincos of the z-line kernels (common.cuh sincos_fast) against the
    oracle's libm, for phases dt H up to 20 rad (every config stays below: <= 1e-12), up to 3e4 rad (fast reduction,
    many quadrants) and beyond 2^30 rad, where the kernel switches to the library routine.  The two sides add the
    terms of H in different orders, so theta itself differs by an ulp: the bound scales with theta.  (8, 8, 100) has
    no z-line kernel: the generic K5 with the library's sincos."""
    dt, g = 0.01, 50.0
    psi = inputs.random_state(shape, 41)
    nmax = float(np.max(np.abs(psi) ** 2))
    psi *= np.sqrt(theta_max / (dt * g * nmax))                    # the largest phase is ~ theta_max
    args = (*shape, 0.3, 0.25, 0.2, dt, 1.0, 0.7, 1.3, g, 0.0, 1)  # gdd = 0: the phase is dt (V + g |psi|^2)
    G, O = gpu.Dgpe(*args), oracle.Oracle(*args)
    amp = float(np.max(np.abs(psi)))
    tol = max(1e-12, 16 * np.finfo(float).eps * theta_max * amp) if theta_max > 20.0 else 1e-12 * max(1.0, amp)
    t, a = dev(psi), psi.copy()
    G.nonlinear(t)
    O.nonlinear(a)
    assert np.max(np.abs(t.cpu().numpy() - a)) <= tol
    t, a = dev(psi), psi.copy()
    assert G.step(t, 1) == O.step(a, 1) == 0
    assert np.max(np.abs(t.cpu().numpy() - a)) <= tol
    assert abs(G.norm(t) / O.norm(a) - 1.0) <= 1e-12               # |exp(-i theta)| = 1 whatever theta


def test_real_time_huge_and_non_finite_phases(gpu, oracle):
    """One point with a phase of 5e299 rad: far beyond the fast reduction, so the kernel must have taken the library
    routine there -- its result is still a pure rotation (|psi'| = |psi| to rounding; the fast reduction would return
    garbage) -- while every other point of the field keeps its 1e-12 parity.  And an overflowing density (inf) gives
    NaN on both sides, as sin(inf) does."""
    shape = (8, 8, 64)
    args = (*shape, 0.3, 0.25, 0.2, 0.01, 1.0, 0.7, 1.3, 50.0, 0.0, 1)
    psi = inputs.random_state(shape, 42)
    psi[3, 4, 20] = 1e150
    G, O = gpu.Dgpe(*args), oracle.Oracle(*args)
    t, a = dev(psi), psi.copy()
    G.nonlinear(t)
    O.nonlinear(a)
    got = t.cpu().numpy()
    assert abs(abs(got[3, 4, 20]) / 1e150 - 1.0) <= 1e-14 and abs(abs(a[3, 4, 20]) / 1e150 - 1.0) <= 1e-14
    got[3, 4, 20] = a[3, 4, 20] = 0.0
    assert np.max(np.abs(got - a)) <= 1e-12
    psi[3, 4, 20] = 1e200                                           # |psi|^2 = inf: theta = inf
    t, a = dev(psi), psi.copy()
    G.nonlinear(t)
    O.nonlinear(a)
    got = t.cpu().numpy()
    assert np.isnan(got[3, 4, 20].real) and np.isnan(a[3, 4, 20].real)


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("shape", [(512, 512, 20), (512, 8, 64), (8, 512, 64), (512, 12, 18)])
def test_fft_pair_kernel_agrees(gpu, oracle, shape, mode):
    """K2 / K3 / K4 at 512 points as k_fft_pair (two tiles per SM in different phases; the default for K3) against the
    one-tile kernels, and both against the oracle's Phi: whole and ragged last tiles ((nz/2+1) = 11, 33, 10 bins; 12 * 10
    = 120 flattened columns), fewer tiles than SMs and more, odd tile counts per CTA."""
    args = (*shape, 0.3, 0.25, 0.2, 0.004, 1.0, 0.7, 1.3, 5.0, 3.0, mode)
    psi = inputs.random_state(shape, 29) * 0.2
    ref = oracle.Oracle(*args).dipolar(np.ascontiguousarray(psi.real ** 2 + psi.imag ** 2))
    out = []
    for opt in ({"tma_pair": 0}, {"tma_pair": 1}, None):
        G = gpu.Dgpe(*args, options=opt)
        phi = G.dipolar(dev(psi)).cpu().numpy()
        assert np.max(np.abs(phi - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref))), opt
        t = dev(psi)
        G.step(t, 4)
        out.append(t.cpu().numpy())
    assert np.max(np.abs(out[0] - out[1])) <= 1e-13 and np.max(np.abs(out[0] - out[2])) <= 1e-13


def test_handles_of_different_sizes_alive_together(gpu, oracle):
    """The shared-memory opt-in of a kernel is per process and device, not per handle: creating a small
    handle must not lower the limit a larger live handle launches with -- generic kernels (972 = 2^2 3^5 has no
    specialised kernel), the observables' K5, and the specialised ones."""
    big_shape, small_shape = (8, 8, 972), (8, 8, 8)
    phys = (0.3, 0.25, 0.2, 0.004, 1.0, 0.7, 1.3, 5.0, 3.0, 0)
    big = gpu.Dgpe(*big_shape, *phys)
    psi = inputs.random_state(big_shape, 31) * 0.3
    t = dev(psi)
    big.step(t, 1)
    small = gpu.Dgpe(*small_shape, *phys)
    ts = dev(inputs.random_state(small_shape, 32) * 0.3)
    small.step(ts, 1)
    small.chempot(ts)
    # the large handle still launches: step, observables, dipolar
    big.step(t, 1)
    a = psi.copy()
    O = oracle.Oracle(*big_shape, *phys)
    O.step(a, 2)
    assert np.max(np.abs(t.cpu().numpy() - a)) <= TOL_1
    assert abs(big.chempot(t) - O.chempot(a)) <= TOL_OBS * abs(O.chempot(a))
    ref = O.dipolar(np.ascontiguousarray(a.real ** 2 + a.imag ** 2))
    assert np.max(np.abs(big.dipolar(t).cpu().numpy() - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    # and the same with the specialised 512-point kernels next to a 64-point handle
    big2 = gpu.Dgpe(512, 8, 8, *phys)
    t2 = dev(inputs.random_state((512, 8, 8), 33) * 0.3)
    big2.step(t2, 1)
    gpu.Dgpe(64, 8, 8, *phys).step(dev(inputs.random_state((64, 8, 8), 34) * 0.3), 1)
    assert big2.step(t2, 1) == gpu.OK


def test_create_reports_the_error_code(gpu):
    with pytest.raises(gpu.DgpeError) as e:
        gpu.Dgpe(8, 8, 10, 0.1, 0.1, 0.1, 0.01, 1.0, 1.0, 1.0, 1.0, 1.0, gpu.IMAG_RPSI)      # nz = 10: no z-line kernel
    assert e.value.code == gpu.ERR_UNSUPPORTED
    with pytest.raises(gpu.DgpeError) as e:
        gpu.Dgpe(8, 8, 17, 0.1, 0.1, 0.1, 0.01, 1.0, 1.0, 1.0, 1.0, 1.0, 0)
    assert e.value.code == gpu.ERR_ARG


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("nx", [384, 480, 512, 640])
def test_k3_tma_pipeline_agrees(gpu, oracle, nx, mode):
    """K3 (FFT_x, Udd~, IFFT_x) has a thread-loading and a TMA-pipelined kernel (the default from nx = 640 up,
    DESIGN.md section 6): each forced in turn gives the same Phi, and that Phi is the oracle's."""
    shape = (nx, 12, 64)            # 12 * 33 = 396 flattened (ky, kz) columns: a ragged last tile (396 = 49 * 8 + 4)
    args = (*shape, 0.3, 0.25, 0.2, 0.004, 1.0, 0.7, 1.3, 5.0, 3.0, mode)
    psi = inputs.random_state(shape, 23) * 0.3
    ref = oracle.Oracle(*args).dipolar(np.ascontiguousarray(psi.real ** 2 + psi.imag ** 2))
    out = []
    for val in (0, 1):
        G = gpu.Dgpe(*args, options={"tma_k3": val})
        out.append(G.dipolar(dev(psi)).cpu().numpy())
        assert np.max(np.abs(out[-1] - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref))), val
        t = dev(psi)
        G.step(t, 3)
        out.append(t.cpu().numpy())
    assert np.max(np.abs(out[0] - out[2])) <= 1e-13
    assert np.max(np.abs(out[1] - out[3])) <= 1e-13


def test_two_handles_on_two_streams(gpu):
    """Handles are independent: two of them stepping different states on two non-default streams at once
    give bit for bit what each gives alone on the default stream (CUDA graph replays included)."""
    cfg = inputs.CONFIGS["C1"]
    psi0 = inputs.initial_state(cfg)
    alone = []
    for seed_scale in (1.0, 0.5):
        t = dev(psi0 * seed_scale)
        gpu.Dgpe(*cfg.create_args()).step(t, 6)
        alone.append(t)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    G1, G2 = gpu.Dgpe(*cfg.create_args(), stream=s1), gpu.Dgpe(*cfg.create_args(), stream=s2)
    a, b = dev(psi0), dev(psi0 * 0.5)
    torch.cuda.synchronize()
    for _ in range(2):                      # 3 + 3 steps, interleaved calls
        G1.step(a, 3)
        G2.step(b, 3)
    G1.synchronize()
    G2.synchronize()
    ref = []
    for seed_scale in (1.0, 0.5):           # the same 3 + 3 call pattern alone (imaginary time renormalises per call)
        t = dev(psi0 * seed_scale)
        H = gpu.Dgpe(*cfg.create_args())
        H.step(t, 3)
        H.step(t, 3)
        ref.append(t)
    assert torch.equal(a, ref[0]) and torch.equal(b, ref[1])
    assert float((a - alone[0]).abs().max()) <= 1e-13


def test_bitwise_repeatable(gpu):
    cfg = inputs.CONFIGS["C1"]
    psi0 = inputs.initial_state(cfg)
    G = gpu.Dgpe(*cfg.create_args())
    a, b = dev(psi0), dev(psi0)
    G.step(a, 5)
    G.step(b, 5)
    assert torch.equal(a, b)


# ------------------------------------------------------------------------------------------------
# full BASELINE sizes, in the launch configuration bench.py times (512^3, C4 handle)
# ------------------------------------------------------------------------------------------------

@pytest.fixture(scope="module")
def c4(gpu):
    cfg = inputs.CONFIGS["C4"]
    return cfg, gpu.Dgpe(*cfg.create_args())


def test_fullsize_dipolar_plane_wave_closed_form(gpu, c4):
    """n = 1 + sum a_m cos(q_m.r + p_m), q_m grid wave vectors  =>  Phi = sum Udd~(q_m) a_m cos(...)
    exactly (pin P4), at 512^3 through the production kernels K1-K5."""
    cfg, G = c4
    nx, ny, nz = cfg.shape
    L = [n * d for n, d in zip(cfg.shape, cfg.d)]
    x, y, z = [torch.from_numpy(inputs.coords(n, d)).cuda() for n, d in zip(cfg.shape, cfg.d)]
    waves = [((3, 0, 0), 0.11, 0.3), ((0, 0, 5), 0.07, 1.1), ((2, -7, 1), 0.05, 2.0), ((-100, 31, 255), 0.02, 0.5),
             ((0, 256, 0), 0.01, 0.0)]
    dens = torch.ones(cfg.shape, dtype=torch.float64, device="cuda")
    phi_ref = torch.zeros_like(dens)
    for m, amp, ph in waves:
        q = [2 * np.pi * mi / Li for mi, Li in zip(m, L)]
        udd = (4 * np.pi / 3) * (3 * q[2] ** 2 / (q[0] ** 2 + q[1] ** 2 + q[2] ** 2) - 1)
        w = torch.cos(q[0] * x[:, None, None] + q[1] * y[None, :, None] + q[2] * z[None, None, :] + ph)
        dens += amp * w
        phi_ref += udd * amp * w
        del w
    psi = torch.sqrt(dens).to(torch.complex128)
    phi = G.dipolar(psi)
    assert float((phi - phi_ref).abs().max()) <= 1e-12
    del phi, phi_ref, dens, psi
    torch.cuda.empty_cache()


def test_fullsize_sweeps_sampled_lines(gpu, oracle, c4):
    """At 512^3 each sweep is compared, on 64 sampled lines per axis, with the oracle's solve of the
    same lines (the oracle sweeps a 512 x 8 x 8 array holding the sampled lines)."""
    cfg, G = c4
    n = 512
    gen = torch.Generator(device="cuda").manual_seed(11)
    psi = torch.randn(cfg.shape, dtype=torch.float64, device="cuda", generator=gen).to(torch.complex128)
    psi += 1j * torch.randn(cfg.shape, dtype=torch.float64, device="cuda", generator=gen)
    rng = np.random.default_rng(12)
    for axis in range(3):
        out = psi.clone()
        G.sweep(out, axis)
        ia, ib = rng.integers(0, n, 64), rng.integers(0, n, 64)
        ia[:4], ib[:4] = [0, 0, n - 1, n - 1], [0, n - 1, 0, n - 1]        # include edge lines
        sel = (torch.from_numpy(ia).cuda(), torch.from_numpy(ib).cuda())
        if axis == 0:
            lin, lout = psi[:, sel[0], sel[1]], out[:, sel[0], sel[1]]             # (512, 64)
        elif axis == 1:
            lin, lout = psi[sel[0], :, sel[1]].T, out[sel[0], :, sel[1]].T
        else:
            lin, lout = psi[sel[0], sel[1], :].T, out[sel[0], sel[1], :].T
        d = cfg.d[axis]
        O = oracle.Oracle(n, 8, 8, d, 1.0, 1.0, cfg.dt, 1, 1, 1, 0.0, 0.0, cfg.mode)
        a = np.ascontiguousarray(lin.cpu().numpy().reshape(n, 8, 8))
        O.sweep(a, 0)
        assert np.max(np.abs(lout.cpu().numpy().reshape(n, 8, 8) - a)) <= TOL_1, axis
        del out
    del psi
    torch.cuda.empty_cache()


def test_fullsize_step_properties(gpu, c4):
    """Literal C4 at 512^3 (the configuration bench.py times): one imaginary-time step returns unit
    norm; with g = gdd = 0 the harmonic ground state is a fixed point of the normalised step up to the
    O(dt, dx^2) splitting error, and mu -> (gamma+nu+lambda)/2 (BJ:north_star check 3)."""
    cfg, G = c4
    psi = dev(inputs.initial_state(cfg))
    assert G.step(psi, 1) == gpu.OK
    assert abs(G.norm(psi) - 1.0) <= 1e-13
    assert bool(torch.isfinite(torch.view_as_real(psi)).all())
    for face in (psi[0], psi[-1], psi[:, 0], psi[:, -1], psi[:, :, 0], psi[:, :, -1]):
        assert float(face.abs().max()) == 0.0
    del psi
    torch.cuda.empty_cache()
    free = inputs.Config("C4-free", cfg.shape, cfg.d, cfg.dt, cfg.trap, 0.0, 0.0, 0, 1, 4, cfg.gauss, noise=0.0)
    G0 = gpu.Dgpe(*free.create_args())
    p0 = dev(inputs.initial_state(free))
    p1 = p0.clone()
    G0.step(p1, 20)
    assert float((p1 - p0).abs().max()) <= 2e-3 * float(p0.abs().max())
    mu = G0.chempot(p1)
    assert abs(mu - 0.5 * sum(cfg.trap)) <= 0.5 * sum(w * w * d * d / 16 for w, d in zip(cfg.trap, cfg.d)) + 5e-3
    assert abs(mu - G0.energy(p1)) <= 1e-12        # no interaction: mu == E


# ------------------------------------------------------------------------------------------------
# BJ:configs[4] at its full size (768 x 768 x 384, real time): the 768- and 384-point kernels in the
# launch configuration bench.py --config C5 times
# ------------------------------------------------------------------------------------------------

def test_fullsize_c5_sweeps_dipolar_and_norm(gpu, oracle):
    cfg = inputs.CONFIGS["C5"]
    nx, ny, nz = cfg.shape
    G = gpu.Dgpe(*cfg.create_args())
    gen = torch.Generator(device="cuda").manual_seed(31)
    psi = torch.randn(cfg.shape, dtype=torch.float64, device="cuda", generator=gen).to(torch.complex128)
    psi += 1j * torch.randn(cfg.shape, dtype=torch.float64, device="cuda", generator=gen)
    rng = np.random.default_rng(32)
    # (c) each sweep on 64 sampled lines per axis (edge lines included) against the oracle's solve
    for axis in range(3):
        n = cfg.shape[axis]
        na, nb = [cfg.shape[a] for a in range(3) if a != axis]
        out = psi.clone()
        G.sweep(out, axis)
        ia, ib = rng.integers(0, na, 64), rng.integers(0, nb, 64)
        ia[:4], ib[:4] = [0, 0, na - 1, na - 1], [0, nb - 1, 0, nb - 1]
        sel = (torch.from_numpy(ia).cuda(), torch.from_numpy(ib).cuda())
        if axis == 0:
            lin, lout = psi[:, sel[0], sel[1]], out[:, sel[0], sel[1]]
        elif axis == 1:
            lin, lout = psi[sel[0], :, sel[1]].T, out[sel[0], :, sel[1]].T
        else:
            lin, lout = psi[sel[0], sel[1], :].T, out[sel[0], sel[1], :].T
        O = oracle.Oracle(n, 8, 8, cfg.d[axis], 1.0, 1.0, cfg.dt, 1, 1, 1, 0.0, 0.0, cfg.mode)
        a = np.ascontiguousarray(lin.cpu().numpy().reshape(n, 8, 8))
        O.sweep(a, 0)
        assert np.max(np.abs(lout.cpu().numpy().reshape(n, 8, 8) - a)) <= TOL_1, axis
        del out
    del psi
    torch.cuda.empty_cache()
    # (a) Phi of plane-wave densities against the closed form (pin P4) through K1-K5
    L = [n * d for n, d in zip(cfg.shape, cfg.d)]
    x, y, z = [torch.from_numpy(inputs.coords(n, d)).cuda() for n, d in zip(cfg.shape, cfg.d)]
    dens = torch.ones(cfg.shape, dtype=torch.float64, device="cuda")
    phi_ref = torch.zeros_like(dens)
    for m, amp, ph in [((3, 0, 0), 0.11, 0.3), ((0, 0, 5), 0.07, 1.1), ((2, -7, 1), 0.05, 2.0), ((-300, 31, 191), 0.02, 0.5),
                       ((0, 384, 0), 0.01, 0.0)]:
        q = [2 * np.pi * mi / Li for mi, Li in zip(m, L)]
        udd = (4 * np.pi / 3) * (3 * q[2] ** 2 / (q[0] ** 2 + q[1] ** 2 + q[2] ** 2) - 1)
        w = torch.cos(q[0] * x[:, None, None] + q[1] * y[None, :, None] + q[2] * z[None, None, :] + ph)
        dens += amp * w
        phi_ref += udd * amp * w
        del w
    psi = torch.sqrt(dens).to(torch.complex128)
    del dens
    phi = G.dipolar(psi)
    assert float((phi - phi_ref).abs().max()) <= 1e-12
    del phi, phi_ref, psi
    torch.cuda.empty_cache()
    # the literal config: real time conserves the norm (BJ:north_star check 4) over 10 steps of the seeded state
    psi = dev(inputs.initial_state(cfg))
    n0 = G.norm(psi)
    assert G.step(psi, 10) == gpu.OK
    assert abs(G.norm(psi) - n0) <= 1e-12
    for face in (psi[0], psi[-1], psi[:, 0], psi[:, -1], psi[:, :, 0], psi[:, :, -1]):
        assert float(face.abs().max()) == 0.0
