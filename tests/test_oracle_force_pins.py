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


# ------------------------------------------------------------------ row f2, second half: d E_L / d R_a (eq. 4)

def test_basis_third_derivatives_by_finite_differences():
    """Hessian = finite differences of the gradient, gradient of the Laplacian = finite differences of the Laplacian."""
    sysm = qi.random_molecule(2, 3, 4, 4, seed=3)              # s, p and d shells
    osys = oracle.OracleSystem(sysm)
    rng = np.random.default_rng(1)
    pairs = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    h = 1e-5
    for _ in range(3):
        r = np.array(sysm.atoms_xyz)[rng.integers(sysm.n_atoms)] + 0.7 * rng.standard_normal(3)
        hess, glap = osys.basis_eval_d3(r)
        for k, (a, b) in enumerate(pairs):
            rp, rm = r.copy(), r.copy()
            rp[b] += h
            rm[b] -= h
            fd = (osys.basis_eval(rp)[1][a] - osys.basis_eval(rm)[1][a]) / (2 * h)
            np.testing.assert_allclose(hess[k], fd, rtol=1e-6, atol=1e-8)
        for d in range(3):
            rp, rm = r.copy(), r.copy()
            rp[d] += h
            rm[d] -= h
            fd = (osys.basis_eval(rp)[2] - osys.basis_eval(rm)[2]) / (2 * h)
            np.testing.assert_allclose(glap[d], fd, rtol=1e-6, atol=1e-7)
        np.testing.assert_allclose(hess[0] + hess[1] + hess[2], osys.basis_eval(r)[2], rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("which", ["water", "molecule"])
def test_deloc_dR_matches_finite_differences_of_the_local_energy(which):
    if which == "water":
        sysm = qi.make_system(0)
        R = qi.initial_positions(sysm, 0, [3])[0]
    else:
        sysm = qi.random_molecule(2, 3, 4, 4, seed=11)
        R = qi.initial_positions(sysm, 0, [1])[0]
    osys = oracle.OracleSystem(sysm)
    w = osys.walker(R)
    for t in range(2):
        w.sweep(5, 0, t, 0.02)
    Rw = w.positions()
    f = w.deloc_dR()
    assert f.shape == (sysm.n_atoms, 3)
    h = 1e-5
    for a in range(sysm.n_atoms):
        for d in range(3):
            ep = oracle.OracleSystem(_displaced(sysm, a, d, +h)).walker(Rw).eloc()[0]
            em = oracle.OracleSystem(_displaced(sysm, a, d, -h)).walker(Rw).eloc()[0]
            fd = (ep - em) / (2 * h)
            assert f[a, d] == pytest.approx(fd, rel=5e-6, abs=5e-6), (a, d)


def test_deloc_dR_translation_sum_rule():
    """E_L is unchanged when nuclei and electrons move together: sum_a dE_L/dR_a = - sum_i grad_i E_L."""
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    R = qi.initial_positions(sysm, 0, [7])[0]
    f = osys.walker(R).deloc_dR().sum(axis=0)
    h = 1e-5
    tot = np.zeros(3)
    for d in range(3):
        Rp, Rm = R.copy(), R.copy()
        Rp[:, d] += h
        Rm[:, d] -= h
        tot[d] = (osys.walker(Rp).eloc()[0] - osys.walker(Rm).eloc()[0]) / (2 * h)
    np.testing.assert_allclose(f, -tot, rtol=5e-6, atol=5e-6)


def test_deloc_dR_atom_subset_is_the_same_numbers():
    sysm = qi.random_molecule(2, 3, 4, 4, seed=11)
    w = oracle.OracleSystem(sysm).walker(qi.initial_positions(sysm, 0, [1])[0])
    full = w.deloc_dR()
    assert np.array_equal(w.deloc_dR([4, 0, 2]), full[[4, 0, 2]])
