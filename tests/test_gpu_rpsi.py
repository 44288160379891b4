"""GPU parity tests (-m gpu) of DGPE_IMAG_RPSI, the real-valued imaginary-time path (SURVEY section 8f
NEXT-2; include/dgpe.h): psi is nx*ny*nz plain doubles.  The oracle has no such mode and needs none: every
factor of its imaginary-time step is real, so its complex psi keeps an exactly zero imaginary part for real
input (pinned in tests/test_oracle_pins.py) and the reference for the real path is the real part of the
oracle's DGPE_IMAG result on the same input.  Same tolerances as tests/test_gpu_parity.py (BJ:north_star)."""
import numpy as np
import pytest
import torch

from paper_1610_05329_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12
TOL_100 = 1e-10
TOL_OBS = 1e-10
RPSI = 2


@pytest.fixture(scope="module")
def gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1610_05329_b200 import binding
    binding.lib()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def pair(gpu, oracle, shape, d, dt, trap, g, gdd):
    return (gpu.Dgpe(*shape, *d, dt, *trap, g, gdd, RPSI), oracle.Oracle(*shape, *d, dt, *trap, g, gdd, 0))


def real_state(shape, seed):
    """Unstructured O(1) real field with zero faces (the real part of the seeded complex stage input)."""
    return np.ascontiguousarray(inputs.random_state(shape, seed).real)


def cx(a):
    return np.ascontiguousarray(a.astype(np.complex128))


# every specialised z length (the real path needs one), lane teams (nz <= 512 powers of two), whole-warp lines,
# first radix 5/6/3 plans, nz/2 odd (ragged complex columns in the x/y sweeps), TMA-fed x/y sweeps, thin boxes
RPSI_SHAPES = [(8, 8, 64), (12, 18, 128), (6, 9, 160), (16, 24, 192), (48, 96, 128), (8, 12, 240), (9, 4, 250),
               (8, 500, 250), (8, 12, 256), (8, 8, 320), (8, 384, 384), (8, 8, 480), (12, 8, 500), (16, 8, 512),
               (8, 8, 640), (4, 8, 768), (768, 8, 64), (16, 768, 128), (64, 64, 64)]


@pytest.mark.parametrize("shape", RPSI_SHAPES)
def test_rpsi_stage_parity(gpu, oracle, shape):
    G, O = pair(gpu, oracle, shape, (0.3, 0.25, 0.2), 0.01, (1.0, 0.7, 1.3), 5.0, 3.0)
    psi = real_state(shape, 3) * 0.3
    # (a) dipolar mean field
    phi = G.dipolar(dev(psi)).cpu().numpy()
    ref = O.dipolar(np.ascontiguousarray(psi ** 2))
    assert np.max(np.abs(phi - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    # (a)+(b) nonlinear exponential
    t, a = dev(psi), cx(psi)
    G.nonlinear(t)
    O.nonlinear(a)
    assert np.all(a.imag == 0)
    assert np.max(np.abs(t.cpu().numpy() - a.real)) <= TOL_1
    # (c) each sweep
    for axis in range(3):
        t, a = dev(psi), cx(psi)
        G.sweep(t, axis)
        O.sweep(a, axis)
        out = t.cpu().numpy()
        assert np.all(a.imag == 0)
        assert np.max(np.abs(out - a.real)) <= TOL_1, axis
        sl = [slice(None)] * 3
        for end in (0, -1):
            sl[axis] = end
            assert np.all(out[tuple(sl)] == 0)
    # observables
    t, a = dev(psi), cx(psi)
    got = [G.norm(t), *G.rms(t), *G.energy_terms(t), G.chempot(t), G.energy(t)]
    exp = [O.norm(a), *O.rms(a), *O.energy_terms(a), O.chempot(a), O.energy(a)]
    for x, y in zip(got, exp):
        assert abs(x - y) <= TOL_OBS * max(1.0, abs(y))
    assert torch.equal(t, dev(psi))                  # observables leave psi alone
    # one full step
    t, a = dev(psi), cx(psi)
    assert G.step(t, 1) == O.step(a, 1) == 0
    assert np.all(a.imag == 0)
    assert np.max(np.abs(t.cpu().numpy() - a.real)) <= TOL_1


@pytest.mark.parametrize("dt", [0.5, 5.0, 40.0])
def test_rpsi_sweeps_with_large_r(gpu, oracle, dt):
    """r up to 250: the z-line kernel and the x/y kernels read the global Thomas tables and look back over
    many chunks (the kernel-parameter tables only hold once the factors have converged)."""
    shape = (8, 384, 128)
    G, O = pair(gpu, oracle, shape, (0.3, 0.25, 0.2), dt, (1.0, 1.0, 1.0), 0.0, 0.0)
    psi = real_state(shape, 5)
    for axis in range(3):
        t, a = dev(psi), cx(psi)
        G.sweep(t, axis)
        O.sweep(a, axis)
        assert np.max(np.abs(t.cpu().numpy() - a.real)) <= 1e-12 * (1 + dt), axis


def run_both(gpu, oracle, cfg, checkpoints):
    psi0 = np.ascontiguousarray(inputs.initial_state(cfg).real)
    args = list(cfg.create_args())
    assert args[-1] == 0, "imaginary-time configs only"
    G, O = gpu.Dgpe(*args[:-1], RPSI), oracle.Oracle(*args)
    t, a = dev(psi0), cx(psi0)
    done, out = 0, []
    for cp in checkpoints:
        rc_g, rc_o = G.step(t, cp - done), O.step(a, cp - done)
        done = cp
        assert rc_g == rc_o
        assert np.all(a.imag == 0)
        err = float(np.max(np.abs(t.cpu().numpy() - a.real)))
        og = [G.norm(t), G.chempot(t), G.energy(t), *G.rms(t)]
        orf = [O.norm(a), O.chempot(a), O.energy(a), *O.rms(a)]
        out.append((cp, err, og, orf))
    return out, t, a


def test_rpsi_c1_full_config_1_and_100_steps(gpu, oracle):
    """BJ:configs[0] (64^3, 100 imaginary-time steps) through the real-valued path."""
    res, _, _ = run_both(gpu, oracle, inputs.CONFIGS["C1"], [1, 10, 100])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100), (cp, err)
        for x, y in zip(og, orf):
            assert abs(x - y) <= TOL_OBS * max(1.0, abs(y)), (og, orf)
        assert abs(og[0] - 1.0) <= 1e-13


def test_rpsi_c2_128cubed_1_and_20_steps(gpu, oracle):
    res, _, _ = run_both(gpu, oracle, inputs.CONFIGS["C2"], [1, 20])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100), (cp, err)
        for x, y in zip(og, orf):
            assert abs(x - y) <= TOL_OBS * max(1.0, abs(y)), (og, orf)


def test_rpsi_c4_physics_scaled_and_status(gpu, oracle):
    """BJ:configs[3] physics on a 64^3 box: smooth window, then the same status of the long call."""
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (64, 64, 64))
    res, t, a = run_both(gpu, oracle, cfg, [1, 10])
    for cp, err, og, orf in res:
        assert err <= (TOL_1 if cp == 1 else TOL_100), (cp, err)
    args = list(cfg.create_args())
    G, O = gpu.Dgpe(*args[:-1], RPSI), oracle.Oracle(*args)
    assert G.step(t, 190) == O.step(a, 190)


def test_rpsi_matches_complex_gpu_path_and_host_path(gpu):
    """The real path against the library's own complex path (same kernels' arithmetic on zero imaginary
    parts), the host-buffer call, bit-repeatability."""
    cfg = inputs.CONFIGS["C1"]
    psi0 = np.ascontiguousarray(inputs.initial_state(cfg).real)
    args = list(cfg.create_args())
    Gr, Gc = gpu.Dgpe(*args[:-1], RPSI), gpu.Dgpe(*args)
    r, c = dev(psi0), dev(cx(psi0))
    Gr.step(r, 10)
    Gc.step(c, 10)
    assert float(c.imag.abs().max()) == 0.0
    assert float((r - c.real).abs().max()) <= 1e-13
    r2 = dev(psi0)
    Gr.step(r2, 10)
    assert torch.equal(r, r2)
    hp = torch.from_numpy(psi0.copy()).pin_memory()
    assert Gr.step_host(hp, 10) == gpu.OK
    assert torch.equal(hp, r.cpu())
    assert Gr.bytes_per_step < Gc.bytes_per_step


def test_rpsi_rejections(gpu):
    with pytest.raises(gpu.DgpeError) as e:
        gpu.Dgpe(8, 8, 96, 0.3, 0.3, 0.3, 0.01, 1, 1, 1, 1.0, 1.0, RPSI)       # 96 is not a specialised z length
    assert "nz" in str(e.value)
    G = gpu.Dgpe(8, 8, 64, 0.3, 0.3, 0.3, 0.01, 1, 1, 1, 1.0, 1.0, RPSI)
    with pytest.raises(TypeError):
        G.step(torch.zeros((8, 8, 64), dtype=torch.complex128, device="cuda"), 1)
    z = torch.zeros((8, 8, 64), dtype=torch.float64, device="cuda")
    assert G.step(z, 1) == gpu.ERR_NONFINITE
    assert G.step(z, 0) == gpu.OK


def test_rpsi_fullsize_512cubed(gpu, oracle):
    """C4's grid (512^3) in the launch configuration `bench.py --config C4r` times: plane-wave Phi closed
    form (pin P4), each sweep on 64 sampled lines against the oracle, unit norm and zero faces after a step."""
    cfg = inputs.CONFIGS["C4"]
    args = list(cfg.create_args())
    G = gpu.Dgpe(*args[:-1], RPSI)
    n = 512
    L = [m * d for m, d in zip(cfg.shape, cfg.d)]
    x, y, z = [torch.from_numpy(inputs.coords(m, d)).cuda() for m, d in zip(cfg.shape, cfg.d)]
    dens = torch.ones(cfg.shape, dtype=torch.float64, device="cuda")
    phi_ref = torch.zeros_like(dens)
    for m, amp, ph in [((3, 0, 0), 0.11, 0.3), ((0, 0, 5), 0.07, 1.1), ((2, -7, 1), 0.05, 2.0), ((-100, 31, 255), 0.02, 0.5)]:
        q = [2 * np.pi * mi / Li for mi, Li in zip(m, L)]
        udd = (4 * np.pi / 3) * (3 * q[2] ** 2 / (q[0] ** 2 + q[1] ** 2 + q[2] ** 2) - 1)
        w = torch.cos(q[0] * x[:, None, None] + q[1] * y[None, :, None] + q[2] * z[None, None, :] + ph)
        dens += amp * w
        phi_ref += udd * amp * w
        del w
    phi = G.dipolar(torch.sqrt(dens))
    assert float((phi - phi_ref).abs().max()) <= 1e-12
    del phi, phi_ref, dens
    torch.cuda.empty_cache()
    gen = torch.Generator(device="cuda").manual_seed(11)
    psi = torch.randn(cfg.shape, dtype=torch.float64, device="cuda", generator=gen)
    rng = np.random.default_rng(12)
    for axis in range(3):
        out = psi.clone()
        G.sweep(out, axis)
        ia, ib = rng.integers(0, n, 64), rng.integers(0, n, 64)
        ia[:4], ib[:4] = [0, 0, n - 1, n - 1], [0, n - 1, 0, n - 1]
        sel = (torch.from_numpy(ia).cuda(), torch.from_numpy(ib).cuda())
        if axis == 0:
            lin, lout = psi[:, sel[0], sel[1]], out[:, sel[0], sel[1]]
        elif axis == 1:
            lin, lout = psi[sel[0], :, sel[1]].T, out[sel[0], :, sel[1]].T
        else:
            lin, lout = psi[sel[0], sel[1], :].T, out[sel[0], sel[1], :].T
        O = oracle.Oracle(n, 8, 8, cfg.d[axis], 1.0, 1.0, cfg.dt, 1, 1, 1, 0.0, 0.0, 0)
        a = cx(lin.cpu().numpy().reshape(n, 8, 8))
        O.sweep(a, 0)
        assert np.max(np.abs(lout.cpu().numpy().reshape(n, 8, 8) - a.real)) <= TOL_1, axis
        del out
    del psi
    torch.cuda.empty_cache()
    psi = dev(np.ascontiguousarray(inputs.initial_state(cfg).real))
    assert G.step(psi, 1) == gpu.OK
    assert abs(G.norm(psi) - 1.0) <= 1e-13
    assert bool(torch.isfinite(psi).all())
    for face in (psi[0], psi[-1], psi[:, 0], psi[:, -1], psi[:, :, 0], psi[:, :, -1]):
        assert float(face.abs().max()) == 0.0
