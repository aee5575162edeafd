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


# ------------------------------------------------------------------ second half: d E_L / d R_a (eq. 4)

@pytest.mark.parametrize("cfg,W,T,k,flags", [(0, 20, 3, 1, 0), (0, 20, 3, 2, 2), (1, 4, 1, 32, 0), ("rand", 9, 2, 2, 2)])
def test_deloc_dR_matches_oracle(cfg, W, T, k, flags):
    if cfg == "rand":
        sysm = qi.random_molecule(3, 4, 6, 6, seed=4)
        pos = qi.initial_positions(sysm, 0, range(W))
        seed, tau = 99, 0.01
    else:
        wl = qi.make_workload(cfg)
        sysm, pos, seed, tau = wl.system, wl.positions(0, W), wl.seed, wl.tau
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, seed, flags=flags)
    qb.qmc_sweep(gw, T, tau, k)
    de, dp = (x.cpu().numpy() for x in qb.qmc_get_deloc_dR(gw))
    gpos = qb.qmc_get_positions(gw).cpu().numpy()
    osys = oracle.OracleSystem(sysm)
    assert de.shape == dp.shape == (W, sysm.n_atoms, 3)
    alone = qb.qmc_get_dlogpsi_dR(gw).cpu().numpy()
    # the first half from the shared C A^-1 product and radial sums: the same numbers as the call of its own (to rounding:
    # the two kernels contract their multiply-adds differently)
    assert np.abs(alone - dp).max() <= 1e-12 * max(1.0, np.abs(alone).max())
    for n in range(W):
        ow = osys.walker(gpos[n])
        ref = ow.deloc_dR()
        # the trace terms carry cond(A) twice (X = A^-1 B A^-1): 1e-8 of the largest component
        assert np.abs(de[n] - ref).max() < 1e-8 * max(1.0, np.abs(ref).max()), (n, np.abs(de[n] - ref).max(), np.abs(ref).max())
        refp = ow.dlogpsi_dR()
        assert np.abs(dp[n] - refp).max() < 1e-9 * max(1.0, np.abs(refp).max()), n


def test_deloc_dR_is_the_finite_difference_of_the_gpu_local_energy():
    """Independent of the oracle: displace one nucleus (a new system on the GPU) and difference the GPU's own E_L."""
    import copy
    wl = qi.make_workload(0)
    sysm = wl.system
    W = 6
    pos = wl.positions(0, W)
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, wl.seed)
    de = qb.qmc_get_deloc_dR(gw, with_dlogpsi=False)[0].cpu().numpy()
    h = 1e-5
    for a in range(sysm.n_atoms):
        for d in range(3):
            e = []
            for sgn in (+1, -1):
                s2 = copy.copy(sysm)
                xyz = np.array(sysm.atoms_xyz, dtype=np.float64, copy=True)
                xyz[a, d] += sgn * h
                s2.atoms_xyz = xyz
                g2 = qb.qmc_init_from(s2)
                e.append(qb.qmc_get_eloc(qb.qmc_walkers_create(g2, pos, wl.seed))[0].cpu().numpy())
            np.testing.assert_allclose(de[:, a, d], (e[0] - e[1]) / (2 * h), rtol=5e-6, atol=5e-5)


def test_deloc_dR_host_output_and_odd_sizes():
    import torch
    sysm = qi.random_molecule(5, 7, 11, 11, seed=21)
    W = 7
    pos = qi.initial_positions(sysm, 0, range(W))
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, 5, flags=2)
    qb.qmc_sweep(gw, 1, 0.01, 3)
    out = torch.empty((W, sysm.n_atoms, 3), dtype=torch.float64)               # host buffer
    de = qb.qmc_get_deloc_dR(gw, out=out, with_dlogpsi=False)[0].numpy()
    gpos = qb.qmc_get_positions(gw).cpu().numpy()
    osys = oracle.OracleSystem(sysm)
    for n in range(W):
        ref = osys.walker(gpos[n]).deloc_dR()
        assert np.abs(de[n] - ref).max() < 1e-8 * max(1.0, np.abs(ref).max()), n


def test_config2_full_size_forces_and_nlpp_sampled():
    """Rows f2 and f3 at the size and in the launch configuration bench.py times (256-water config, 256 walkers): the
    oracle does two sampled walkers, three sampled atoms for dE_L/dR_a and d ln|Psi|/dR_a, and a pseudopotential that
    is switched on for six atoms only (the oracle then has a few dozen quadrature pairs per walker to do)."""
    from concurrent.futures import ThreadPoolExecutor
    wl = qi.make_workload(2)
    sysm = wl.system
    atoms = [0, 1, 767]
    ecp = qi.make_ecp(sysm)
    rc = np.zeros(sysm.n_atoms)
    rc[[0, 1, 2, 300, 301, 767]] = 2.0
    ecp.rcut = rc
    g = qb.qmc_init_from(sysm)
    qb.qmc_set_ecp(g, ecp)
    gw = qb.qmc_walkers_create(g, wl.positions(), wl.seed)
    de, dp = (x.cpu().numpy() for x in qb.qmc_get_deloc_dR(gw))
    vnl, n_pairs = qb.qmc_get_vnl(gw)
    vnl = vnl.cpu().numpy()
    assert n_pairs > 0
    osys = oracle.OracleSystem(sysm)
    sample = [0, 255]

    def one(n):
        ow = osys.walker(wl.positions(n, n + 1)[0])
        return n, ow.deloc_dR(atoms), ow.dlogpsi_dR()[atoms], ow.vnl(ecp, wl.seed, n, 0)
    with ThreadPoolExecutor(max_workers=2) as ex:
        res = list(ex.map(one, sample))
    for n, ref_e, ref_p, ref_v in res:
        # cond(A) up to ~1e6 at N_s = 1024 (reading A26) enters the trace terms twice
        assert np.abs(de[n][atoms] - ref_e).max() < 1e-7 * max(1.0, np.abs(ref_e).max()), (n, de[n][atoms], ref_e)
        assert np.abs(dp[n][atoms] - ref_p).max() < 1e-8 * max(1.0, np.abs(ref_p).max()), n
        assert vnl[n] == pytest.approx(ref_v, rel=1e-8, abs=1e-9), n
