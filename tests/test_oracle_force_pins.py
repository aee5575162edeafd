"""Pin of the oracle's d ln|Psi| / d R_a (row f2, first half; the paper's eq. 3, with lambda a nuclear
coordinate): central finite differences of from-scratch log|Psi| when a nucleus is displaced together with the basis
functions centred on it and its electron-nucleus Jastrow term.  CPU only."""
import copy

import numpy as np
import pytest

import oracle
import qmc_inputs as qi


def _displaced(system, atom, d, h):
    s = copy.copy(system)
    xyz = np.array(system.atoms_xyz, dtype=np.float64, copy=True)
    xyz[atom, d] += h
    s.atoms_xyz = xyz
    return s


@pytest.mark.parametrize("which", ["water", "molecule"])
def test_dlogpsi_dR_matches_finite_differences(which):
    if which == "water":
        sysm = qi.make_system(0)
        R = qi.initial_positions(sysm, 0, [3])[0]
    else:
        sysm = qi.random_molecule(2, 3, 4, 4, seed=11)
        R = qi.initial_positions(sysm, 0, [1])[0]
    osys = oracle.OracleSystem(sysm)
    w = osys.walker(R)
    for t in range(2):                       # a state with updated inverses, not just the LU one
        w.sweep(5, 0, t, 0.02)
    Rw = w.positions()
    g = w.dlogpsi_dR()
    assert g.shape == (sysm.n_atoms, 3)
    h = 1e-5
    for a in range(sysm.n_atoms):
        for d in range(3):
            lp = oracle.OracleSystem(_displaced(sysm, a, d, +h)).walker(Rw).logpsi()
            lm = oracle.OracleSystem(_displaced(sysm, a, d, -h)).walker(Rw).logpsi()
            assert lp[1] == lm[1]
            fd = (lp[0] - lm[0]) / (2 * h)
            assert g[a, d] == pytest.approx(fd, rel=2e-6, abs=2e-7), (a, d)


def test_dlogpsi_dR_translation_sum_rule():
    """Moving every nucleus AND every electron by the same vector leaves Psi unchanged, so
    sum_a d ln|Psi|/dR_a = - sum_i grad_i ln|Psi|; the right-hand side from finite differences over the electrons."""
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    R = qi.initial_positions(sysm, 0, [7])[0]
    g = osys.walker(R).dlogpsi_dR().sum(axis=0)
    h = 1e-5
    tot = np.zeros(3)
    for d in range(3):
        Rp, Rm = R.copy(), R.copy()
        Rp[:, d] += h
        Rm[:, d] -= h
        tot[d] = (osys.walker(Rp).logpsi()[0] - osys.walker(Rm).logpsi()[0]) / (2 * h)
    np.testing.assert_allclose(g, -tot, rtol=2e-6, atol=2e-7)
