"""Row f3 on the GPU against the oracle (-m gpu): non-local pseudopotential energy of every walker through the C ABI."""
import math

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


@pytest.mark.parametrize("cfg,W,T,k,flags,scale", [(0, 40, 3, 1, 0, 1.0), (0, 40, 3, 2, 2, 2.0), (1, 6, 1, 32, 0, 1.0),
                                                   ("rand", 9, 2, 2, 2, 1.5)])
def test_vnl_matches_oracle(cfg, W, T, k, flags, scale):
    if cfg == "rand":
        sysm = qi.random_molecule(3, 4, 6, 6, seed=4)
        pos = qi.initial_positions(sysm, 0, range(W))
        seed, tau, first = 99, 0.01, 0
    else:
        wl = qi.make_workload(cfg)
        sysm, pos, seed, tau, first = wl.system, wl.positions(0, W), wl.seed, wl.tau, 0
    ecp = qi.make_ecp(sysm)
    ecp.rcut[:] *= scale
    g = qb.qmc_init_from(sysm)
    qb.qmc_set_ecp(g, ecp)
    gw = qb.qmc_walkers_create(g, pos, seed, flags=flags)
    qb.qmc_sweep(gw, T, tau, k)                      # sweep counter = T: the rotations of step T
    v, n_pairs = qb.qmc_get_vnl(gw)
    v = v.cpu().numpy()
    gpos = qb.qmc_get_positions(gw).cpu().numpy()
    osys = oracle.OracleSystem(sysm)
    xyz = np.array(sysm.atoms_xyz)
    count = 0
    for n in range(W):
        ref = osys.walker(gpos[n]).vnl(ecp, seed, first + n, T)
        d = np.linalg.norm(gpos[n][:, None, :] - xyz[None, :, :], axis=2)
        count += int((d < ecp.rcut[None, :]).sum())
        assert v[n] == pytest.approx(ref, rel=1e-9, abs=1e-9), n
    assert n_pairs == count and count > 0
    assert np.std(v) > 0


@pytest.mark.parametrize("l,m", [(0, 0), (1, 1), (2, 3)])
def test_one_orbital_atom_closed_form_on_gpu(l, m):
    sysm = qi.one_orbital_atom(l, m)
    ecp = qi.Ecp(np.array([0, 0, 0], np.int32), np.array([0, 1, 2], np.int32), np.array([3.0, -1.5, 0.8]),
                 np.array([0.9, 0.6, 0.4]), np.array([2.5]))
    rng = np.random.default_rng(17 + l)
    pos = rng.standard_normal((32, 1, 3)) * 0.5
    pos = pos[np.linalg.norm(pos[:, 0], axis=1) < 2.4]
    g = qb.qmc_init_from(sysm)
    qb.qmc_set_ecp(g, ecp)
    gw = qb.qmc_walkers_create(g, pos, 3)
    v = qb.qmc_get_vnl(gw)[0].cpu().numpy()
    r = np.linalg.norm(pos[:, 0], axis=1)
    np.testing.assert_allclose(v, ecp.ch_beta[l] * np.exp(-ecp.ch_alpha[l] * r * r), rtol=1e-10)


def test_vnl_edge_cases():
    import torch
    wl = qi.make_workload(0)
    sysm = wl.system
    pos = wl.positions(0, 5)
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, wl.seed)
    with pytest.raises(qb.QmcError):
        qb.qmc_get_vnl(gw)                                         # no pseudopotential set
    ecp = qi.make_ecp(sysm)
    none = qi.Ecp(ecp.ch_atom, ecp.ch_l, ecp.ch_beta, ecp.ch_alpha, np.full(sysm.n_atoms, 1e-9))
    qb.qmc_set_ecp(g, none)
    v, n = qb.qmc_get_vnl(gw)
    assert n == 0 and float(v.abs().max()) == 0.0                  # nothing inside the cut-off
    qb.qmc_set_ecp(g, ecp)                                         # replaced table; host output buffer
    out = torch.empty(5, dtype=torch.float64)
    v2, n2 = qb.qmc_get_vnl(gw, out=out)
    assert n2 > 0 and v2.abs().max() > 0
    v3, _ = qb.qmc_get_vnl(gw)
    assert np.array_equal(v2.numpy(), v3.cpu().numpy())            # same sweep counter, same rotations: reproducible
    bad = qi.Ecp(np.array([99], np.int32), np.array([0], np.int32), np.array([1.0]), np.array([1.0]), ecp.rcut)
    with pytest.raises(qb.QmcError):
        qb.qmc_set_ecp(g, bad)
