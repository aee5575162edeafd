"""Pins for the CPU oracle: every part of oracle/qmc_oracle.c is checked against something other than
itself -- published known-answer vectors, closed forms, finite differences, numpy.linalg routines,
brute force on tiny inputs, and invariants (BASELINE.json north_star).  CPU only."""
import math
import os

import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from qmc_inputs import System

HERE = os.path.dirname(os.path.abspath(__file__))


def one_shell_system(l, alpha, coef, Z=0.0, n_up=1, C=None, b_en=1.0, centre=(0.0, 0.0, 0.0)):
    nb = 2 * l + 1
    if C is None:
        C = np.zeros((nb, n_up))
        C[0, 0] = 1.0
    return System(name="one_shell", atoms_xyz=np.array([centre], float), Z=np.array([Z]),
                  shell_atom=np.array([0], np.int32), shell_l=np.array([l], np.int32),
                  shell_nprim=np.array([len(alpha)], np.int32), shell_prim_offset=np.array([0], np.int32),
                  alpha=np.asarray(alpha, float), coef=np.asarray(coef, float), n_basis=nb, n_up=n_up, n_dn=0,
                  C_up=np.asarray(C, float), C_dn=np.zeros((nb, 0)), b_en=b_en,
                  electron_atom=np.zeros(n_up, np.int32))


# ------------------------------------------------------------------ RNG

def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(w[0:4], w[4:6])
        assert out.tolist() == w[6:10]
        out_ld = oracle.philox4x32_10(w[0:4], w[4:6], long_double=True)
        assert out_ld.tolist() == w[6:10]


def test_uniform_mapping_exact_and_keyed():
    # U = (2*(x>>12)+1) * 2^-53 with x = (w0<<32)|w1 of block 0: recompute from the raw Philox words
    seed = (0x12345678 << 32) | 0x9ABCDEF0
    for (w, s, e) in [(0, 0, 0), (5, 7, 11), (4095, 99, 2047)]:
        U = oracle.move_uniforms(seed, w, s, e)
        key = [seed & 0xFFFFFFFF, seed >> 32]
        for blk in range(3):
            o = oracle.philox4x32_10([w, s, e, blk], key)
            x = (int(o[0]) << 32) | int(o[1])
            assert U[2 * blk] == (2 * (x >> 12) + 1) * 2.0 ** -53
            if blk < 2:
                x = (int(o[2]) << 32) | int(o[3])
                assert U[2 * blk + 1] == (2 * (x >> 12) + 1) * 2.0 ** -53
        assert np.all((U > 0) & (U < 1))
        assert np.all((U * 2.0 ** 53) % 2 == 1)  # odd integers: never 0, never 1
    # different (walker, step, electron) -> different streams
    a = oracle.move_uniforms(seed, 1, 2, 3)
    assert not np.array_equal(a, oracle.move_uniforms(seed, 2, 1, 3))
    assert not np.array_equal(a, oracle.move_uniforms(seed, 1, 3, 2))
    assert not np.array_equal(a, oracle.move_uniforms(seed + 1, 1, 2, 3))


def test_box_muller_definition_and_moments():
    seed = 7948
    U = oracle.move_uniforms(seed, 3, 4, 5)
    chi, u = oracle.move_variates(seed, 3, 4, 5)
    r1, r2 = math.sqrt(-2 * math.log(U[0])), math.sqrt(-2 * math.log(U[2]))
    np.testing.assert_allclose(chi, [r1 * math.cos(2 * math.pi * U[1]), r1 * math.sin(2 * math.pi * U[1]),
                                     r2 * math.cos(2 * math.pi * U[3])], rtol=1e-15, atol=1e-15)
    assert u == U[4]
    n = 60000
    xs = np.array([np.append(*oracle.move_variates(seed, w, 0, 0)) for w in range(n)])
    assert np.all(np.abs(xs[:, :3].mean(0)) < 5 / math.sqrt(n))
    assert np.all(np.abs(xs[:, :3].var(0) - 1) < 5 * math.sqrt(2 / n))
    assert abs(np.mean(xs[:, 0] * xs[:, 1])) < 5 / math.sqrt(n)
    assert abs(xs[:, 3].mean() - 0.5) < 5 / math.sqrt(12 * n)


# ------------------------------------------------------------------ basis functions

def _fd_grad_lap(f, r, h=1e-4):
    r = np.asarray(r, float)
    f0 = f(r)
    g = np.zeros((3,) + f0.shape)
    lap = np.zeros_like(f0)
    for d in range(3):
        e = np.zeros(3)
        e[d] = h
        fp, fm = f(r + e), f(r - e)
        g[d] = (fp - fm) / (2 * h)
        lap += (fp - 2 * f0 + fm) / (h * h)
    return g, lap


@pytest.mark.parametrize("cfg", [0])
def test_basis_gradient_laplacian_vs_finite_differences(cfg):
    sysm = qi.make_system(cfg)
    osys = oracle.OracleSystem(sysm)
    rng = np.random.default_rng(1)
    for _ in range(6):
        r = sysm.atoms_xyz[rng.integers(sysm.n_atoms)] + rng.standard_normal(3) * 0.7
        phi, grad, lap = osys.basis_eval(r)
        g_fd, lap_fd = _fd_grad_lap(lambda x: osys.basis_eval(x)[0], r, h=1e-4)
        scale = np.abs(phi).max() + 1e-30
        assert np.abs(grad - g_fd).max() < 1e-6 * max(1.0, np.abs(grad).max())
        # second differences: error ~ h^2 f'''' + eps/h^2
        assert np.abs(lap - lap_fd).max() < 1e-5 * max(1.0, np.abs(lap).max()), (np.abs(lap - lap_fd).max(), scale)


def test_basis_single_s_primitive_closed_form():
    al, d = 0.8, 1.7
    osys = oracle.OracleSystem(one_shell_system(0, [al], [d], centre=(0.3, -0.2, 0.1)))
    r = np.array([1.0, 0.4, -0.6])
    x = r - np.array([0.3, -0.2, 0.1])
    t = x @ x
    phi, grad, lap = osys.basis_eval(r)
    assert phi[0] == pytest.approx(d * math.exp(-al * t), rel=1e-15)
    np.testing.assert_allclose(grad[:, 0], -2 * al * x * d * math.exp(-al * t), rtol=1e-14)
    assert lap[0] == pytest.approx((4 * al * al * t - 6 * al) * d * math.exp(-al * t), rel=1e-14)


def test_angular_factors_are_harmonic_and_ordered():
    # alpha = 0, coef = 1: Phi = S_lm exactly; lap S = 0, x.grad S = l S, and the listed polynomials
    r = np.array([0.7, -1.3, 0.45])
    x, y, z = r
    s3 = math.sqrt(3.0)
    expect = {0: [1.0], 1: [x, y, z],
              2: [s3 * x * y, s3 * y * z, z * z - 0.5 * (x * x + y * y), s3 * x * z, 0.5 * s3 * (x * x - y * y)]}
    for l in (0, 1, 2):
        osys = oracle.OracleSystem(one_shell_system(l, [0.0], [1.0]))
        phi, grad, lap = osys.basis_eval(r)
        np.testing.assert_allclose(phi, expect[l], rtol=1e-15)
        np.testing.assert_allclose(lap, 0, atol=1e-15)
        np.testing.assert_allclose(r @ grad, l * phi, rtol=1e-14, atol=1e-15)


def test_contracted_functions_have_unit_self_overlap_and_shell_is_orthogonal():
    # 3-D quadrature of Phi_a Phi_b in spherical coordinates (composite Gauss-Legendre in r, Gauss-Legendre
    # in cos(theta), trapezoid in phi: exact for the degree-4 angular polynomials): pins the Racah
    # normalisation of the angular factors together with the generator's contraction normalisation
    #
    edges = np.concatenate([[0.0], 0.05 * 2.0 ** np.arange(0, 9)])  # 0 .. 12.8 bohr, geometric panels
    gx, gw = np.polynomial.legendre.leggauss(14)
    rr = np.concatenate([0.5 * (b - a) * gx + 0.5 * (a + b) for a, b in zip(edges[:-1], edges[1:])])
    rw = np.concatenate([0.5 * (b - a) * gw for a, b in zip(edges[:-1], edges[1:])])
    ct, cw = np.polynomial.legendre.leggauss(6)
    ph = 2 * np.pi * np.arange(10) / 10
    for l in (0, 1, 2):
        alpha = np.array([0.35, 0.9, 2.2])
        coef = qi.contract_normalised(alpha, [0.3, 0.8, 0.5], l)
        centre = np.array([0.2, -0.1, 0.3])
        osys = oracle.OracleSystem(one_shell_system(l, alpha, coef, centre=tuple(centre)))
        nf = 2 * l + 1
        S = np.zeros((nf, nf))
        for r, wr in zip(rr, rw):
            for c, wc in zip(ct, cw):
                st = math.sqrt(1 - c * c)
                for f in ph:
                    v = osys.basis_eval(centre + r * np.array([st * math.cos(f), st * math.sin(f), c]))[0]
                    S += wr * r * r * wc * (2 * np.pi / len(ph)) * np.outer(v, v)
        np.testing.assert_allclose(S, np.eye(nf), atol=1e-10)


def test_mo_rows_are_the_contraction_Ct_phi():
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    r = np.array([0.4, 0.9, -0.3])
    phi, grad, lap = osys.basis_eval(r)
    for spin, Cm in ((0, sysm.C_up), (1, sysm.C_dn)):
        rows = osys.mo_rows(spin, r)
        np.testing.assert_allclose(rows[0], Cm.T @ phi, rtol=1e-13, atol=1e-15)
        for d in range(3):
            np.testing.assert_allclose(rows[1 + d], Cm.T @ grad[d], rtol=1e-13, atol=1e-14)
        np.testing.assert_allclose(rows[4], Cm.T @ lap, rtol=1e-13, atol=1e-13)
    # brute-force double loop on one entry (index order / transposition)
    j = 3
    assert osys.mo_rows(0, r)[0, j] == pytest.approx(sum(sysm.C_up[l, j] * phi[l] for l in range(sysm.n_basis)), rel=1e-13)


# ------------------------------------------------------------------ linear algebra

@pytest.mark.parametrize("n", [1, 2, 3, 5, 8, 40])
def test_lu_inverse_vs_numpy(n):
    rng = np.random.default_rng(n)
    A = rng.standard_normal((n, n))
    rc, Ainv, lad, sg = oracle.lu_inverse(A)
    assert rc == 0
    np.testing.assert_allclose(Ainv, np.linalg.inv(A), rtol=1e-9, atol=1e-11)
    s_np, l_np = np.linalg.slogdet(A)
    assert sg == int(s_np) and lad == pytest.approx(l_np, abs=1e-12)


def test_lu_inverse_flags_singular():
    A = np.array([[1.0, 2.0], [2.0, 4.0]])
    assert oracle.lu_inverse(A)[0] == -3
    assert oracle.lu_inverse(np.zeros((3, 3)))[0] == -3


@pytest.mark.parametrize("n", [2, 4, 8])
def test_determinant_ratio_and_sherman_morrison_vs_explicit(n):
    rng = np.random.default_rng(100 + n)
    A = rng.standard_normal((n, n))
    Ainv = np.linalg.inv(A)  # Ainv[j][p]
    for p in range(n):
        v = rng.standard_normal(n)
        A2 = A.copy()
        A2[p] = v
        new_inv, rho = oracle.sherman_morrison(Ainv, p, v)
        assert rho == pytest.approx(np.linalg.det(A2) / np.linalg.det(A), rel=1e-11)
        np.testing.assert_allclose(new_inv, np.linalg.inv(A2), rtol=1e-8, atol=1e-10)


@pytest.mark.parametrize("n,m", [(4, 1), (6, 3), (8, 8), (24, 7)])
def test_delayed_rank_k_update_vs_direct_inverse(n, m):
    rng = np.random.default_rng(n * 31 + m)
    A0 = rng.standard_normal((n, n)) + 2 * np.eye(n)
    rows = rng.permutation(n)[:m]
    V = rng.standard_normal((m, n))
    A1 = A0.copy()
    A1[rows] = V
    rc, out, det = oracle.delayed_update(np.linalg.inv(A0), rows, V)
    assert rc == 0
    np.testing.assert_allclose(out, np.linalg.inv(A1), rtol=1e-8, atol=1e-10)
    s1, l1 = np.linalg.slogdet(A1)
    s0, l0 = np.linalg.slogdet(A0)
    assert det[0] == s1 * s0 and det[1] == pytest.approx(l1 - l0, abs=1e-10)  # det S = det A'/det A0
    # and the same result by m successive Sherman-Morrison steps; det S = product of the rho's
    Ainv = np.linalg.inv(A0)
    prod = 1.0
    for a in range(m):
        Ainv, rho = oracle.sherman_morrison(Ainv, rows[a], V[a])
        prod *= rho
    np.testing.assert_allclose(Ainv, out, rtol=1e-8, atol=1e-10)
    assert prod == pytest.approx(det[0] * math.exp(det[1]), rel=1e-9)


# ------------------------------------------------------------------ Jastrow

def _two_electron_system(same_spin, Z=0.0):
    s = one_shell_system(0, [0.5], [1.0], Z=Z, n_up=1)
    if same_spin:
        s.n_up, s.n_dn = 2, 0
        s.C_up, s.C_dn = np.zeros((1, 2)), np.zeros((1, 0))
    else:
        s.n_up, s.n_dn = 1, 1
        s.C_up, s.C_dn = np.ones((1, 1)), np.ones((1, 1))
    return s


def test_jastrow_cusps():
    # u'(0) = a: 1/2 for antiparallel, 1/4 for parallel spins, -Z at a nucleus (BASELINE.json configs[0])
    for same, a in ((False, 0.5), (True, 0.25)):
        osys = oracle.OracleSystem(_two_electron_system(same))
        eps = 1e-7
        R = np.array([[5.0, 5.0, 5.0], [5.0 + eps, 5.0, 5.0]])
        J, g, lap = osys.jastrow(R)
        assert g[1, 0] == pytest.approx(a, rel=1e-6) and g[0, 0] == pytest.approx(-a, rel=1e-6)
    osys = oracle.OracleSystem(_two_electron_system(False, Z=3.0))
    R = np.array([[1e-7, 0.0, 0.0], [40.0, 0.0, 0.0]])
    J, g, lap = osys.jastrow(R)
    assert g[0, 0] == pytest.approx(-3.0 - 0.5 / 41 ** 2, rel=1e-5)


def test_jastrow_value_gradient_laplacian():
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    R = qi.initial_positions(sysm, 0, [3])[0]
    J, g, lap = osys.jastrow(R)
    # value by an independent numpy double sum
    Jn = 0.0
    ne = sysm.n_elec
    for i in range(ne):
        for k in range(i + 1, ne):
            a = 0.25 if (i < sysm.n_up) == (k < sysm.n_up) else 0.5
            r = np.linalg.norm(R[i] - R[k])
            Jn += a * r / (1 + r)
        for I in range(sysm.n_atoms):
            r = np.linalg.norm(R[i] - sysm.atoms_xyz[I])
            Jn += -sysm.Z[I] * r / (1 + r)
    assert J == pytest.approx(Jn, rel=1e-13)
    for i in (0, 4, 7):
        def f(x):
            R2 = R.copy()
            R2[i] = x
            return np.array(osys.jastrow(R2)[0])
        g_fd, lap_fd = _fd_grad_lap(f, R[i], h=1e-4)
        np.testing.assert_allclose(g[i], g_fd, rtol=1e-6, atol=1e-7)
        assert lap[i] == pytest.approx(float(lap_fd), rel=1e-4, abs=1e-5)


# ------------------------------------------------------------------ wave function invariants

def test_hydrogen_local_energy_is_minus_half_everywhere():
    osys = oracle.OracleSystem(qi.hydrogen_atom())
    rng = np.random.default_rng(0)
    for _ in range(20):
        r = rng.standard_normal(3) * rng.uniform(0.05, 4.0)
        w = osys.walker(r[None, :])
        e, k = w.eloc()
        assert e == pytest.approx(-0.5, abs=1e-13)
        assert w.logpsi()[0] == pytest.approx(-np.linalg.norm(r), abs=1e-14)
    # zero variance along a trajectory, and <r> -> 3/2 for |exp(-r)|^2 (weak sampling check of the
    # drift-diffusion + accept/reject rule: a wrong sign in the Green's-function ratio biases it)
    res = oracle.run_crowd(qi.hydrogen_atom(), rng.standard_normal((64, 1, 3)), 11, range(64), 0, 1500, 0.05, threads=1)
    assert np.abs(res["eloc"] + 0.5).max() < 1e-12
    rs = []
    ws = [osys.walker(p) for p in res["positions"]]
    for t in range(400):
        for n, w in enumerate(ws):
            w.sweep(11, n, 1500 + t, 0.05)
            rs.append(np.linalg.norm(w.positions()[0]))
    assert np.mean(rs) == pytest.approx(1.5, abs=0.06)


def test_single_gaussian_kinetic_energy_closed_form():
    al = 0.6
    s = one_shell_system(0, [al], [1.0], Z=0.0)
    osys = oracle.OracleSystem(s)
    for r in ([0.3, 0.2, -0.5], [1.5, -1.0, 0.7]):
        w = osys.walker(np.array([r]))
        e, k = w.eloc()
        r2 = float(np.dot(r, r))
        assert k == pytest.approx(3 * al - 2 * al * al * r2, rel=1e-13)
        assert e == pytest.approx(k, rel=1e-13)  # Z = 0, one electron: V = 0


def test_antisymmetry_under_same_spin_swap():
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    R = qi.initial_positions(sysm, 0, [1])[0]
    w1 = osys.walker(R)
    for (a, b) in ((0, 3), (6, 9)):
        R2 = R.copy()
        R2[[a, b]] = R2[[b, a]]
        w2 = osys.walker(R2)
        (l1, s1), (l2, s2) = w1.logpsi(), w2.logpsi()
        assert l2 == pytest.approx(l1, abs=1e-10) and s2 == -s1
        assert w2.eloc()[0] == pytest.approx(w1.eloc()[0], rel=1e-10)
    # opposite-spin swap is NOT a symmetry of a spin-assigned Slater-Jastrow function
    R3 = R.copy()
    R3[[0, 5]] = R3[[5, 0]]
    assert abs(osys.walker(R3).logpsi()[0] - w1.logpsi()[0]) > 1e-6


def test_log_derivative_identity_eq3():
    # PAPER.md L173 eq. (3): d ln D / d lambda = tr(A^-1 dA/d lambda).  lambda = a coordinate of electron i
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    R = qi.initial_positions(sysm, 0, [2])[0]
    w = osys.walker(R)
    _, gJ, _ = osys.jastrow(R)
    for i in (1, 4, 8):
        spin, p = (0, i) if i < sysm.n_up else (1, i - sysm.n_up)
        rows = osys.mo_rows(spin, R[i])
        g = rows[1:4] @ w.Ainv(spin)[p]  # sum_j grad phi_j(r_i) (A^-1)_{j p}
        assert rows[0] @ w.Ainv(spin)[p] == pytest.approx(1.0, abs=1e-11)  # row p of A times column p of A^-1
        def f(x):
            R2 = R.copy()
            R2[i] = x
            return np.array(osys.walker(R2).logpsi()[0])
        g_fd, _ = _fd_grad_lap(f, R[i], h=1e-5)
        np.testing.assert_allclose(g + gJ[i], g_fd, rtol=2e-5, atol=1e-6)


def test_local_energy_vs_finite_difference_laplacian_of_log_psi():
    # K = -1/2 sum_i [ lap_i ln|Psi| + |grad_i ln|Psi||^2 ] by finite differences of from-scratch log|Psi|
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    R = qi.initial_positions(sysm, 0, [5])[0]
    w = osys.walker(R)
    K = 0.0
    for i in range(sysm.n_elec):
        def f(x):
            R2 = R.copy()
            R2[i] = x
            return np.array(osys.walker(R2).logpsi()[0])
        g, lap = _fd_grad_lap(f, R[i], h=2e-4)
        K += -0.5 * (float(lap) + float(g @ g))
    e, k = w.eloc()
    assert k == pytest.approx(K, rel=2e-5)
    # potential by an independent numpy sum
    V = 0.0
    for i in range(sysm.n_elec):
        for j in range(i + 1, sysm.n_elec):
            V += 1 / np.linalg.norm(R[i] - R[j])
        for I in range(sysm.n_atoms):
            V -= sysm.Z[I] / np.linalg.norm(R[i] - sysm.atoms_xyz[I])
    for I in range(sysm.n_atoms):
        for J in range(I + 1, sysm.n_atoms):
            V += sysm.Z[I] * sysm.Z[J] / np.linalg.norm(sysm.atoms_xyz[I] - sysm.atoms_xyz[J])
    assert e - k == pytest.approx(V, rel=1e-12)


# ------------------------------------------------------------------ the move itself

def test_acceptance_probability_from_first_principles():
    """Replay one sweep electron by electron with quantities the sweep code does not share:
    |Psi|^2 ratio and drifts from finite differences of from-scratch log|Psi| (LU, direct Jastrow sums),
    Green's-function ratio written out.  Pins drift, proposal, rho_D*exp(dJ), Delta, p_acc, the accept
    rule, move order (A10) and the state carried from one electron to the next."""
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    seed, wid, step, tau = 424242, 17, 3, 0.01
    R = qi.initial_positions(sysm, 0, [wid])[0]
    w = osys.walker(R)
    bits, ratio, pacc = w.sweep(seed, wid, step, tau)
    Rc = R.copy()
    n_checked = 0
    for i in range(sysm.n_elec):
        def logpsi_at(x, i=i):
            R2 = Rc.copy()
            R2[i] = x
            return osys.walker(R2).logpsi()
        f = lambda x: np.array(logpsi_at(x)[0])
        G, _ = _fd_grad_lap(f, Rc[i], h=1e-5)
        chi, u = oracle.move_variates(seed, wid, step, i)
        rp = Rc[i] + tau * G + math.sqrt(tau) * chi
        (l0, s0), (l1, s1) = logpsi_at(Rc[i]), logpsi_at(rp)
        if s0 != s1:
            assert bits[i] & 1 == 0 and pacc[i] == 0.0  # fixed node (A7)
            continue
        Gp, _ = _fd_grad_lap(f, rp, h=1e-5)
        fwd = np.sum((rp - Rc[i] - tau * G) ** 2)
        rev = np.sum((Rc[i] - rp - tau * Gp) ** 2)
        p_expect = math.exp(2 * (l1 - l0) + (fwd - rev) / (2 * tau))
        assert pacc[i] == pytest.approx(p_expect, rel=3e-4), i
        assert ratio[i] == pytest.approx(math.exp(l1 - l0), rel=1e-5)
        if abs(u - p_expect) > 1e-3:
            assert bool(bits[i] & 1) == (u < p_expect)
        if bits[i] & 1:
            Rc[i] = rp
        n_checked += 1
    assert n_checked >= 8
    np.testing.assert_allclose(w.positions(), Rc, atol=1e-6)


def test_running_state_matches_from_scratch_after_sweeps():
    for cfg, nsw, wid in ((0, 30, 2), (1, 1, 0)):
        wl = qi.make_workload(cfg)
        sysm = wl.system
        osys = oracle.OracleSystem(sysm)
        w = osys.walker(wl.positions(wid, wid + 1)[0])
        acc = 0
        for t in range(nsw):
            bits, ratio, pacc = w.sweep(wl.seed, wid, t, wl.tau)
            acc += int((bits & 1).sum())
            (la, sg), (lb, sb) = w.logpsi(), w.logpsi_scratch()
            assert sg == sb and la == pytest.approx(lb, rel=1e-12, abs=1e-9)
        assert acc > 0.5 * nsw * sysm.n_elec
        # inverse carried by Sherman-Morrison == inverse of the Slater matrix rebuilt from the positions,
        # and the stored orbital rows are bitwise what a fresh evaluation gives
        Rf = w.positions()
        for spin, e0 in ((0, 0), (1, sysm.n_up)):
            ns = osys.ns(spin)
            A = np.stack([osys.mo_rows(spin, Rf[e0 + p])[0] for p in range(ns)])
            AinvT = w.Ainv(spin)  # [p][j] = (A^-1)[j][p]
            np.testing.assert_allclose(A @ AinvT.T, np.eye(ns), atol=1e-8)
        w2 = osys.walker(Rf)
        assert w2.eloc()[0] == pytest.approx(w.eloc()[0], rel=1e-9)


def test_tie_and_node_flags_and_walker_prefix_independence():
    wl = qi.make_workload(0)
    a = oracle.run_crowd(wl.system, wl.positions(0, 6), wl.seed, range(6), 0, 5, wl.tau, threads=1)
    b = oracle.run_crowd(wl.system, wl.positions(2, 4), wl.seed, range(2, 4), 0, 5, wl.tau, threads=2)
    assert np.array_equal(a["bits"][:, :, 2:4], b["bits"])  # A20: a walker depends only on (seed, w)
    assert np.array_equal(a["positions"][2:4], b["positions"])
    # resume: 2 + 3 sweeps == 5 sweeps (A12: the step counter is global)
    osys = oracle.OracleSystem(wl.system)
    w = osys.walker(wl.positions(1, 2)[0])
    for t in range(5):
        w.sweep(wl.seed, 1, t, wl.tau)
    assert np.array_equal(w.positions(), a["positions"][1])
    assert set(np.unique(a["bits"])) <= {0, 1, 2, 3}
    # a rejected node crossing reports p_acc = 0
    assert np.all(a["pacc"][(a["bits"] & 1) == 1] > 0)


def test_long_double_build_agrees_with_double():
    wl = qi.make_workload(0)
    a = oracle.run_crowd(wl.system, wl.positions(0, 2), wl.seed, range(2), 0, 10, wl.tau, threads=1)
    b = oracle.run_crowd(wl.system, wl.positions(0, 2), wl.seed, range(2), 0, 10, wl.tau, threads=1, long_double=True)
    assert oracle._lib(True).oracle_real_bytes() > 8
    assert np.array_equal(a["bits"] & 1, b["bits"] & 1)
    np.testing.assert_allclose(a["positions"], b["positions"], atol=1e-11)
    np.testing.assert_allclose(a["eloc"], b["eloc"], rtol=1e-10)
