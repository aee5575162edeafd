"""Pins of the oracle's non-local pseudopotential energy (row f3; reading A34).  CPU only.
The quadrature rule against the closed-form sphere integrals of monomials; the energy against closed forms on one-
orbital atoms (the projector on l picks v_l exactly); every wave-function ratio against from-scratch log|Psi|; the
sum against a separately typed Legendre / weight / channel bookkeeping; cut-off and additivity."""
import math

import numpy as np
import pytest

import oracle
import qmc_inputs as qi


def _dfact(n):
    return 1 if n <= 0 else n * _dfact(n - 2)


def test_rotated_icosahedron_integrates_degree_five_exactly():
    """mean over the sphere of x^a y^b z^c = (a-1)!!(b-1)!!(c-1)!!/(a+b+c+1)!! for even a, b, c and 0 otherwise."""
    for el in range(4):
        d = oracle.quadrature_directions(11, 3, 7, el)
        np.testing.assert_allclose(np.linalg.norm(d, axis=1), 1.0, rtol=1e-14)
        for a in range(6):
            for b in range(6 - a):
                for c in range(6 - a - b):
                    got = np.mean(d[:, 0] ** a * d[:, 1] ** b * d[:, 2] ** c)
                    exact = 0.0
                    if a % 2 == 0 and b % 2 == 0 and c % 2 == 0:
                        exact = _dfact(a - 1) * _dfact(b - 1) * _dfact(c - 1) / _dfact(a + b + c + 1)
                    assert got == pytest.approx(exact, abs=2e-15), (a, b, c)
    # degree 6 is NOT integrated exactly (it is a 12-point rule, not more) and rotations differ between electrons
    d0, d1 = oracle.quadrature_directions(11, 3, 7, 0), oracle.quadrature_directions(11, 3, 7, 1)
    assert abs(np.mean(d0[:, 0] ** 6) - 1 / 7) > 1e-4
    assert np.abs(d0 - d1).max() > 1e-3
    assert np.array_equal(d0, oracle.quadrature_directions(11, 3, 7, 0))


def test_rotations_are_uniform_enough():
    """first moments of the rotated first vertex over many counters: mean 0, covariance I/3"""
    v = np.array([oracle.quadrature_directions(5, w, 0, 0)[0] for w in range(4000)])
    assert np.abs(v.mean(axis=0)).max() < 0.03
    np.testing.assert_allclose(v.T @ v / len(v), np.eye(3) / 3, atol=0.02)


@pytest.mark.parametrize("l,m", [(0, 0), (1, 0), (1, 2), (2, 0), (2, 2), (2, 4)])
def test_one_orbital_atom_picks_its_own_channel(l, m):
    """Psi = S_lm(r) f(|r|): the angular projector on l' returns delta_ll' Psi, and the integrand is a polynomial of
    degree 2l <= 4 on the sphere, so the 12-point rule is exact: V_nl = v_l(r) whatever the rotation."""
    sysm = qi.one_orbital_atom(l, m)
    osys = oracle.OracleSystem(sysm)
    ecp = qi.Ecp(np.array([0, 0, 0], np.int32), np.array([0, 1, 2], np.int32), np.array([3.0, -1.5, 0.8]),
                 np.array([0.9, 0.6, 0.4]), np.array([2.5]))
    rng = np.random.default_rng(l * 7 + m)
    for trial in range(4):
        R = rng.standard_normal((1, 3)) * 0.6
        r = np.linalg.norm(R)
        if r >= 2.5:
            continue
        try:
            w = osys.walker(R)
        except ArithmeticError:
            continue
        v = w.vnl(ecp, 99, trial, 5)
        assert v == pytest.approx(ecp.ch_beta[l] * math.exp(-ecp.ch_alpha[l] * r * r), rel=1e-11)


def _legendre(l, c):
    return [1.0, c, 1.5 * c * c - 0.5][l]


@pytest.mark.parametrize("which", ["water", "molecule"])
def test_ratios_from_scratch_and_the_bookkeeping(which):
    if which == "water":
        sysm = qi.make_system(0)
        R = qi.initial_positions(sysm, 0, [2])[0]
    else:
        sysm = qi.random_molecule(2, 3, 4, 4, seed=11)
        R = qi.initial_positions(sysm, 0, [1])[0]
    ecp = qi.make_ecp(sysm)
    ecp.rcut[:] *= 1.6                                     # more pairs inside the cut-off
    osys = oracle.OracleSystem(sysm)
    w = osys.walker(R)
    for t in range(2):
        w.sweep(5, 0, t, 0.02)
    Rw = w.positions()
    seed, wid, step = 31, 4, 9
    v, pi, pI, pts, rat = w.vnl(ecp, seed, wid, step, details=True)
    xyz = np.array(sysm.atoms_xyz)
    # the pair list is exactly the (electron, atom) pairs inside the cut-off, electrons then atoms ascending
    expect = [(i, I) for i in range(sysm.n_elec) for I in range(sysm.n_atoms) if np.linalg.norm(Rw[i] - xyz[I]) < ecp.rcut[I]]
    assert list(zip(pi.tolist(), pI.tolist())) == expect and len(expect) >= 3
    lp0 = w.logpsi_scratch()
    total = 0.0
    for n, (i, I) in enumerate(expect):
        x = Rw[i] - xyz[I]
        r = np.linalg.norm(x)
        dirs = oracle.quadrature_directions(seed, wid, step, i)
        np.testing.assert_allclose(pts[n], xyz[I] + r * dirs, atol=1e-13)
        for q in range(12):
            R2 = Rw.copy()
            R2[i] = pts[n, q]
            lp = osys.walker(R2).logpsi()
            ratio = lp[1] * lp0[1] * math.exp(lp[0] - lp0[0])
            assert rat[n, q] == pytest.approx(ratio, rel=1e-8, abs=1e-10)
            c = float(dirs[q] @ x) / r
            for ch in range(ecp.n_channels):
                if ecp.ch_atom[ch] == I:
                    l = int(ecp.ch_l[ch])
                    total += (2 * l + 1) * ecp.ch_beta[ch] * math.exp(-ecp.ch_alpha[ch] * r * r) * _legendre(l, c) * ratio / 12
    assert v == pytest.approx(total, rel=1e-8)


def test_cutoff_and_additivity():
    sysm = qi.make_system(0)
    ecp = qi.make_ecp(sysm)
    ecp.rcut[:] = 3.0
    osys = oracle.OracleSystem(sysm)
    w = osys.walker(qi.initial_positions(sysm, 0, [5])[0])
    full = w.vnl(ecp, 1, 0, 0)
    # nothing inside the cut-off: zero
    none = qi.Ecp(ecp.ch_atom, ecp.ch_l, ecp.ch_beta, ecp.ch_alpha, np.full(sysm.n_atoms, 1e-6))
    assert w.vnl(none, 1, 0, 0) == 0.0
    # linear in the channels: the sum of one-channel energies is the energy
    parts = 0.0
    for ch in range(ecp.n_channels):
        one = qi.Ecp(ecp.ch_atom[ch:ch + 1], ecp.ch_l[ch:ch + 1], ecp.ch_beta[ch:ch + 1], ecp.ch_alpha[ch:ch + 1], ecp.rcut)
        parts += w.vnl(one, 1, 0, 0)
    assert full == pytest.approx(parts, rel=1e-12)
    # a different step rotates the grids: the energy changes a little (quadrature error), not wildly
    other = w.vnl(ecp, 1, 0, 1)
    assert other != full and abs(other - full) < 0.2 * abs(full) + 0.5
