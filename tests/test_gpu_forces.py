"""Row f2, first half, on the GPU against the oracle (-m gpu): d ln|Psi| / d R_a for every atom and walker."""
import numpy as np
import pytest

import oracle
import qmc_inputs as qi

pytestmark = pytest.mark.gpu

qb = pytest.importorskip("paper_2504_07948_b200")


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    qb.load_library()


@pytest.mark.parametrize("cfg,W,T,k,flags", [(0, 20, 3, 1, 0), (0, 20, 3, 2, 2), (1, 6, 1, 32, 0), ("rand", 9, 2, 2, 2)])
def test_dlogpsi_dR_matches_oracle(cfg, W, T, k, flags):
    if cfg == "rand":
        sysm = qi.random_molecule(3, 4, 6, 6, seed=4)
        pos = qi.initial_positions(sysm, 0, range(W))
        seed, tau = 99, 0.01
    else:
        wl = qi.make_workload(cfg)
        sysm, pos, seed, tau = wl.system, wl.positions(0, W), wl.seed, wl.tau
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, seed, flags=flags)
    qb.qmc_sweep(gw, T, tau, k)                      # inverses carried by the (delayed) updates, not fresh ones
    got = qb.qmc_get_dlogpsi_dR(gw).cpu().numpy()
    gpos = qb.qmc_get_positions(gw).cpu().numpy()
    osys = oracle.OracleSystem(sysm)
    assert got.shape == (W, sysm.n_atoms, 3)
    for n in range(W):
        ref = osys.walker(gpos[n]).dlogpsi_dR()
        assert np.abs(got[n] - ref).max() < 1e-9 * max(1.0, np.abs(ref).max()), n


def test_dlogpsi_dR_host_output_and_sum_rule():
    """sum_a d ln|Psi|/dR_a = - sum_i grad_i ln|Psi| (translation invariance); the right-hand side from finite
    differences of the GPU's own log|Psi| over rigidly shifted electrons."""
    import torch
    wl = qi.make_workload(0)
    pos = wl.positions(0, 4)
    g = qb.qmc_init_from(wl.system)
    gw = qb.qmc_walkers_create(g, pos, wl.seed)
    out = torch.empty((4, wl.system.n_atoms, 3), dtype=torch.float64)          # host buffer
    got = qb.qmc_get_dlogpsi_dR(gw, out=out).numpy().sum(axis=1)
    h = 1e-5
    for d in range(3):
        sh = np.zeros(3)
        sh[d] = h
        lp = qb.qmc_get_logpsi(qb.qmc_walkers_create(g, pos + sh, wl.seed))[0].cpu().numpy()
        lm = qb.qmc_get_logpsi(qb.qmc_walkers_create(g, pos - sh, wl.seed))[0].cpu().numpy()
        np.testing.assert_allclose(got[:, d], -(lp - lm) / (2 * h), rtol=2e-6, atol=2e-7)
