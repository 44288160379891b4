"""GPU test (-m gpu) of dgpe_norm_noalloc, the one entry point that allocates nothing (static device scratch; include/dgpe.h):
its result against the existing path's (dgpe_norm on a handle), on two calls in a row that share the scratch array.
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

from paper_1610_05329_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_OBS = 1e-10          # the observables' tolerance of the other GPU tests (BJ:north_star), relative


@pytest.fixture(scope="module")
def gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1610_05329_b200 import binding
    binding.lib()
    return binding


def test_norm_noalloc_matches_dgpe_norm_on_two_calls_in_a_row(gpu):
    d = (0.3, 0.25, 0.2)
    # two different shapes and states back to back: the second call finds the first call's partials and ticket in the scratch
    cases = [((64, 48, 40), 71, 0.7), ((24, 60, 32), 72, 1.9)]
    psis = [torch.from_numpy(inputs.random_state(shape, seed, zero_faces=False) * amp).cuda() for shape, seed, amp in cases]
    outs = [torch.full((1,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    before = torch.cuda.memory_allocated()
    for psi, out in zip(psis, outs):                                  # no synchronisation in between
        assert gpu.norm_noalloc(psi, *d, out) == gpu.OK
    assert torch.cuda.memory_allocated() == before
    torch.cuda.synchronize()
    for (shape, _, _), psi, out in zip(cases, psis, outs):
        G = gpu.Dgpe(*shape, *d, 0.01, 1.0, 1.0, 1.0, 1.0, 1.0, gpu.IMAG)
        ref = G.norm(psi)                                             # the existing path: k_moments with cudaMalloc'ed scratch
        got = float(out[0])
        assert abs(got - ref) <= TOL_OBS * abs(ref), (shape, got, ref)
        host = float(np.sum(np.abs(psi.cpu().numpy()) ** 2) * d[0] * d[1] * d[2])
        assert abs(got - host) <= 1e-12 * abs(host)
        G.close()
    # the same call again gives the same bits (fixed summation order, scratch fully re-initialised)
    again = torch.zeros(1, dtype=torch.float64, device="cuda")
    assert gpu.norm_noalloc(psis[0], *d, again) == gpu.OK
    torch.cuda.synchronize()
    assert float(again[0]) == float(outs[0][0])


def test_norm_noalloc_rejects_what_does_not_fit_the_static_scratch(gpu):
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    big = torch.zeros((gpu.NOALLOC_MAX_NX + 1, 2, 2), dtype=torch.complex128, device="cuda")
    assert gpu.norm_noalloc(big, 0.1, 0.1, 0.1, out) == gpu.ERR_UNSUPPORTED
    assert "DGPE_NOALLOC_MAX_NX" in gpu.last_error()
    edge = torch.ones((gpu.NOALLOC_MAX_NX, 2, 2), dtype=torch.complex128, device="cuda")      # the maximum itself is accepted
    assert gpu.norm_noalloc(edge, 0.5, 0.5, 0.5, out) == gpu.OK
    torch.cuda.synchronize()
    assert abs(float(out[0]) - gpu.NOALLOC_MAX_NX * 4 * 0.125) <= 1e-12 * gpu.NOALLOC_MAX_NX
    assert gpu.norm_noalloc(edge, 0.5, -0.5, 0.5, out) == gpu.ERR_ARG
    with pytest.raises(TypeError):
        gpu.norm_noalloc(edge.to(torch.complex64), 0.5, 0.5, 0.5, out)
