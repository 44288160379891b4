"""GPU parity tests (-m gpu) of the slab-decomposed step: P ranks emulated on ONE device
(paper_1610_05329_b200/sharded.py LocalComm: the exchanges are device-to-device copies of the same (NX/P) x (NY/P) x NZ blocks an
all-to-all would move), compared element by element with the CPU oracle and with the unsharded CUDA step.  The multi-process
exchange itself is tested on CPU tensors with gloo (tests/test_sharded_gloo.py); no multi-GPU hardware was available."""
import numpy as np
import pytest
import torch

from paper_1610_05329_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1610_05329_b200 import binding
    binding.lib()
    return binding


def slabs_of(psi, P):
    nxl = psi.shape[0] // P
    return [torch.from_numpy(np.ascontiguousarray(psi[p * nxl:(p + 1) * nxl])).cuda() for p in range(P)]


def gather(slabs):
    return torch.cat(slabs, dim=0).cpu().numpy()


# (shape, ranks): cubic and non-cubic, z-line kernels (nz = 64, 128) and generic z (nz = 20, 36), radix 3 and 5,
# thin slabs (nx/P = 2), TMA-sized lines (384, 512) next to short ones
CASES = [((16, 16, 16), 1), ((16, 16, 16), 2), ((16, 16, 16), 4), ((64, 32, 64), 4), ((48, 96, 20), 3), ((30, 20, 36), 5),
         ((32, 64, 128), 8), ((384, 16, 64), 2), ((16, 512, 64), 4),
         ((512, 16, 64), 2)]           # nx = 512: the x pass of the y-slab view runs as k_fft_pair


@pytest.mark.parametrize("shape,P", CASES)
@pytest.mark.parametrize("mode", [0, 1])
def test_sharded_step_matches_oracle_and_unsharded(gpu, oracle, shape, P, mode):
    from paper_1610_05329_b200 import sharded
    args = (*shape, 0.3, 0.25, 0.2, 0.004, 1.0, 0.7, 1.3, 5.0, 3.0, mode)
    psi = inputs.random_state(shape, 51) * 0.2
    S = sharded.ShardedDgpe(*args, sharded.LocalComm(P))
    slabs = slabs_of(psi, P)
    a = psi.copy()
    O = oracle.Oracle(*args)
    G = gpu.Dgpe(*args)
    t = torch.from_numpy(psi.copy()).cuda()
    done = 0
    for cp in (1, 4):
        assert S.step(slabs, cp - done) == O.step(a, cp - done) == G.step(t, cp - done) == 0
        done = cp
        got = gather(slabs)
        assert np.max(np.abs(got - a)) <= (1e-12 if cp == 1 else 1e-10), (shape, P, mode, cp)
        assert np.max(np.abs(got - t.cpu().numpy())) <= 1e-13
    full = torch.from_numpy(gather(slabs)).cuda()
    for og, orf in zip([G.norm(full), G.chempot(full), G.energy(full)], [O.norm(a), O.chempot(a), O.energy(a)]):
        assert abs(og - orf) <= 1e-10 * max(1.0, abs(orf))
    if mode == 0:
        assert abs(G.norm(full) - 1.0) <= 1e-13                 # the norm was summed over the ranks
    S.close()


def test_sharded_c1_config_20_steps(gpu, oracle):
    """BJ:configs[0] (64^3, imaginary time) on 4 emulated ranks, 20 steps."""
    from paper_1610_05329_b200 import sharded
    cfg = inputs.CONFIGS["C1"]
    psi = inputs.initial_state(cfg)
    S = sharded.ShardedDgpe(*cfg.create_args(), sharded.LocalComm(4))
    slabs = slabs_of(psi, 4)
    a = psi.copy()
    O = oracle.Oracle(*cfg.create_args())
    assert S.step(slabs, 20) == O.step(a, 20) == 0
    assert np.max(np.abs(gather(slabs) - a)) <= 1e-10
    S.close()


def test_sharded_rejects_indivisible_grids_and_reports_collapse(gpu):
    from paper_1610_05329_b200 import sharded
    with pytest.raises(ValueError):
        sharded.ShardedDgpe(16, 18, 16, 0.3, 0.3, 0.3, 0.01, 1, 1, 1, 1.0, 1.0, 0, sharded.LocalComm(4))
    S = sharded.ShardedDgpe(16, 16, 16, 0.3, 0.3, 0.3, 0.01, 1, 1, 1, 1.0, 1.0, 0, sharded.LocalComm(2))
    zero = [torch.zeros((8, 16, 16), dtype=torch.complex128, device="cuda") for _ in range(2)]
    assert S.step(zero, 1) == gpu.ERR_NONFINITE                  # zero state: norm 0, as the unsharded step reports it
    with pytest.raises(TypeError):
        S.step([z.to(torch.complex64) for z in zero], 1)
    S.close()
