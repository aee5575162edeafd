"""Pins of the oracle's DMC generation (row f1 of SURVEY 8(f): drift limiter, effective time step, branching weight,
comb reconfiguration) against things other than itself: the literal Umrigar-Nightingale-Runge limiter formula, closed
forms on the hydrogen atom (E_L = -1/2 exactly), every p_acc of a limited-drift sweep recomputed from finite
differences of from-scratch log|Psi|, the weight formula from separately evaluated energies, and the comb's defining
properties by brute force.  CPU only."""
import math

import numpy as np
import pytest

import oracle
import qmc_inputs as qi
from test_oracle_pins import _fd_grad_lap


def _limiter_literal(v2, a, tau):
    """UNR 1993 eq. (35) as printed: (-1 + sqrt(1 + 2 a v^2 tau)) / (a v^2 tau), in extended precision."""
    x = np.longdouble(a) * np.longdouble(v2) * np.longdouble(tau)
    return float((np.sqrt(1 + 2 * x) - 1) / x)


def test_drift_limiter_matches_the_literal_formula_and_its_limits():
    for v2 in (1e-3, 0.3, 7.0, 250.0, 4e4, 1e9):
        for a in (0.5, 1.0):
            for tau in (0.002, 0.01, 0.05):
                assert oracle.drift_limiter_scale(v2, a, tau) == pytest.approx(_limiter_literal(v2, a, tau), rel=1e-13)
    assert oracle.drift_limiter_scale(0.0, 1.0, 0.01) == 1.0
    assert oracle.drift_limiter_scale(1e-12, 1.0, 0.01) == pytest.approx(1.0, abs=1e-13)   # v -> 0: no limiting
    assert oracle.drift_limiter_scale(3.0, 0.0, 0.01) == 1.0                                # a = 0 switches it off (A6)
    # large drift: |vbar| tau -> sqrt(2 tau / a), the displacement can no longer exceed the diffusion length scale
    v2, a, tau = 1e12, 1.0, 0.01
    assert oracle.drift_limiter_scale(v2, a, tau) * math.sqrt(v2) * tau == pytest.approx(math.sqrt(2 * tau / a), rel=1e-4)
    # monotone: the limited speed grows with the raw speed and never exceeds it
    s = [oracle.drift_limiter_scale(v * v, 1.0, 0.01) for v in np.linspace(0.1, 50, 40)]
    assert all(0 < x <= 1 for x in s) and all(b < a for a, b in zip(s, s[1:]))


def test_limiter_off_is_the_plain_sweep_bit_for_bit():
    wl = qi.make_workload(0)
    osys = oracle.OracleSystem(wl.system)
    R = wl.positions(3, 4)[0]
    a, b = osys.walker(R), osys.walker(R)
    for t in range(4):
        ba, ra, pa = a.sweep(wl.seed, 3, t, wl.tau)
        bb, rb, pb, dr2 = b.sweep_limited(wl.seed, 3, t, wl.tau, 0.0)
        assert np.array_equal(ba, bb) and np.array_equal(ra, rb) and np.array_equal(pa, pb)
        assert 0 < dr2[0] <= dr2[1]
    assert np.array_equal(a.positions(), b.positions())


def test_limited_sweep_acceptance_from_first_principles():
    """As test_acceptance_probability_from_first_principles, with the limiter: drifts from finite differences of
    from-scratch log|Psi|, limited by the literal formula, forward and reverse."""
    sysm = qi.make_system(0)
    osys = oracle.OracleSystem(sysm)
    seed, wid, step, tau, a = 9090, 5, 2, 0.02, 1.0
    R = qi.initial_positions(sysm, 0, [wid])[0]
    w = osys.walker(R)
    bits, ratio, pacc, dr2 = w.sweep_limited(seed, wid, step, tau, a)
    Rc = R.copy()
    n_checked, n_limited = 0, 0
    rr_acc = rr_all = 0.0
    for i in range(sysm.n_elec):
        def logpsi_at(x, i=i):
            R2 = Rc.copy()
            R2[i] = x
            return osys.walker(R2).logpsi()
        f = lambda x: np.array(logpsi_at(x)[0])
        G, _ = _fd_grad_lap(f, Rc[i], h=1e-5)
        sG = _limiter_literal(G @ G, a, tau)
        n_limited += sG < 0.9
        G = G * sG
        chi, u = oracle.move_variates(seed, wid, step, i)
        rr = tau * float(chi @ chi)
        rr_all += rr
        rp = Rc[i] + tau * G + math.sqrt(tau) * chi
        (l0, s0), (l1, s1) = logpsi_at(Rc[i]), logpsi_at(rp)
        if s0 != s1:
            assert bits[i] & 1 == 0 and pacc[i] == 0.0
            continue
        Gp, _ = _fd_grad_lap(f, rp, h=1e-5)
        Gp = Gp * _limiter_literal(Gp @ Gp, a, tau)
        fwd = np.sum((rp - Rc[i] - tau * G) ** 2)
        rev = np.sum((Rc[i] - rp - tau * Gp) ** 2)
        p_expect = math.exp(2 * (l1 - l0) + (fwd - rev) / (2 * tau))
        assert pacc[i] == pytest.approx(p_expect, rel=1e-3), i
        if abs(u - p_expect) > 1e-2 * max(1.0, p_expect):
            assert bool(bits[i] & 1) == (u < p_expect)
        if bits[i] & 1:
            Rc[i] = rp
            rr_acc += rr
        n_checked += 1
    assert n_checked >= 8 and n_limited >= 1      # the O electrons near the nucleus have |G| ~ 8: the limiter is active
    np.testing.assert_allclose(w.positions(), Rc, atol=1e-6)
    assert dr2[1] == pytest.approx(rr_all, rel=1e-12) and dr2[0] == pytest.approx(rr_acc, rel=1e-12)


def _tau_eff_from_log(seed, wid, step, tau, bits, n_elec):
    acc = tot = 0.0
    for i in range(n_elec):
        chi, _ = oracle.move_variates(seed, wid, step, i)
        rr = tau * float(chi @ chi)
        tot += rr
        if bits[i] & 1:
            acc += rr
    return tau * acc / tot


def test_hydrogen_weights_are_the_closed_form():
    """Exact trial function exp(-r): E_L = -1/2 at every point, so after any generation
    w = w_old * exp(-tau_eff * (-1/2 - E_T)) with tau_eff fixed by the accept record alone."""
    osys = oracle.OracleSystem(qi.hydrogen_atom())
    rng = np.random.default_rng(5)
    seed, tau, e_t, a = 77, 0.05, -0.45, 1.0
    for wid in range(6):
        w = osys.walker(rng.standard_normal((1, 3)))
        e_old, weight = w.eloc()[0], 1.0
        assert e_old == pytest.approx(-0.5, abs=1e-12)
        expect = 1.0
        for t in range(40):
            bits, e_new, weight, te = w.dmc_generation(seed, wid, t, tau, a, e_t, e_old, weight)
            te_expect = _tau_eff_from_log(seed, wid, t, tau, bits, 1)
            assert te == pytest.approx(te_expect, rel=1e-13, abs=1e-300)
            assert te in (0.0, pytest.approx(tau))        # one electron: the move was accepted or it was not
            assert e_new == pytest.approx(-0.5, abs=1e-10)
            expect *= math.exp(-te_expect * (-0.5 - e_t))
            e_old = e_new
        assert weight == pytest.approx(expect, rel=1e-9)


def test_generation_weight_and_time_step_from_separately_evaluated_pieces():
    wl = qi.make_workload(0)
    sysm = wl.system
    osys = oracle.OracleSystem(sysm)
    seed, tau, e_t, a = wl.seed, wl.tau, -70.0, 1.0
    for wid in (0, 9):
        R = wl.positions(wid, wid + 1)[0]
        w, twin = osys.walker(R), osys.walker(R)
        e_old, weight = w.eloc()[0], 0.8
        for t in range(5):
            bits, e_new, w_new, te = w.dmc_generation(seed, wid, t, tau, a, e_t, e_old, weight)
            # the same sweep through the logging entry point, energies from a walker rebuilt from the positions
            b2, _, _, dr2 = twin.sweep_limited(seed, wid, t, tau, a)
            assert np.array_equal(bits, b2)
            assert te == pytest.approx(_tau_eff_from_log(seed, wid, t, tau, bits, sysm.n_elec), rel=1e-13)
            assert te == pytest.approx(tau * dr2[0] / dr2[1], rel=1e-14)
            e_scratch = osys.walker(w.positions()).eloc()[0]
            assert e_new == pytest.approx(e_scratch, rel=1e-9)
            assert w_new == pytest.approx(weight * math.exp(-te * (0.5 * (e_old + e_scratch) - e_t)), rel=1e-9)
            assert 0 < te <= tau
            e_old, weight = e_new, w_new


# ------------------------------------------------------------------ comb reconfiguration

def _comb_brute(weights, xi):
    """multiplicities by counting, for every walker, the teeth inside its cumulative-weight interval (exact rationals)"""
    from fractions import Fraction
    w = [Fraction(float(x)) for x in weights]
    W, tot = len(w), sum(w)
    teeth = [(Fraction(j) + Fraction(float(xi))) * tot / W for j in range(W)]
    lo, m = Fraction(0), []
    for x in w:
        m.append(sum(1 for t in teeth if lo <= t < lo + x))
        lo += x
    return m


def test_comb_multiplicities_by_brute_force_and_slot_rule():
    rng = np.random.default_rng(12)
    for trial in range(40):
        W = int(rng.integers(2, 40))
        w = rng.gamma(2.0, 0.5, W)
        if trial % 5 == 0:
            w[rng.integers(0, W)] *= 6.0          # one heavy walker: several copies
        xi = float(rng.random())
        src, mult, neww = oracle.comb_reconfigure(w, xi)
        brute = _comb_brute(w, xi)
        # rounding of the cumulative sums can move a tooth across one boundary; away from such ties the counts are equal
        if list(mult) != brute:
            cum = np.cumsum(w)
            teeth = (np.arange(W) + xi) * (cum[-1] / W)
            assert np.min(np.abs(teeth[:, None] - cum[None, :-1])) < 1e-12
            continue
        assert mult.sum() == W and neww == pytest.approx(w.sum() / W, rel=1e-14)
        ideal = W * w / w.sum()
        assert np.all(mult >= np.floor(ideal)) and np.all(mult <= np.ceil(ideal))
        # survivors stay in place; the k-th dead slot takes the k-th extra copy, donors ascending
        assert all(src[k] == k for k in range(W) if mult[k] > 0)
        dead = [k for k in range(W) if mult[k] == 0]
        assert list(src[dead]) == sorted(src[dead])
        assert np.array_equal(np.bincount(src, minlength=W), mult)


def test_comb_is_unbiased_and_trivial_for_equal_weights():
    W = 12
    src, mult, _ = oracle.comb_reconfigure(np.ones(W), 0.37)
    assert np.array_equal(src, np.arange(W)) and np.all(mult == 1)
    rng = np.random.default_rng(3)
    w = rng.gamma(2.0, 0.5, W)
    tot = np.zeros(W)
    n = 4000
    for _ in range(n):
        tot += oracle.comb_reconfigure(w, float(rng.random()))[1]
    np.testing.assert_allclose(tot / n, W * w / w.sum(), atol=0.03)   # E[m_i] = W w_i / sum w


def test_comb_uniform_is_a_philox_word_pair():
    xi = oracle.comb_uniform(7948, 11)
    out = oracle.philox4x32_10([0xFFFFFFFF, 11, 0xFFFFFFFF, 3], [7948, 0])
    x = (int(out[0]) << 32) | int(out[1])
    assert xi == (2 * (x >> 12) + 1) / 2.0 ** 53 and 0.0 < xi < 1.0
    assert oracle.comb_uniform(7948, 12) != xi


# ------------------------------------------------------------------ the run with population control (reading A32)

def test_hydrogen_run_with_population_control_is_the_closed_form():
    """E_L = -1/2 everywhere: the mixed estimator is -1/2 at every reconfiguration, every weight is
    exp(tau (1/2 + E_T)) per accepted move, so the whole E_T trajectory follows from the accept record alone; the slot
    maps are the brute-force comb's on those weights."""
    osys = oracle.OracleSystem(qi.hydrogen_atom())
    rng = np.random.default_rng(9)
    W, G, every, fb, tau, seed = 16, 12, 3, 0.5, 0.08, 314
    walkers = [osys.walker(rng.standard_normal((1, 3))) for _ in range(W)]
    r = oracle.dmc_run(osys, walkers, seed, range(W), 5, G, tau, 1.0, -0.4, every, fb)
    wt, e_t = np.ones(W), -0.4
    n_branch = 0
    for g in range(G):
        assert r["e_trial_log"][g] == pytest.approx(e_t, rel=1e-12)
        wt = wt * np.exp(tau * (r["bits"][g, 0] & 1) * (0.5 + e_t))
        if (g + 1) % every == 0:
            n_branch += 1
            assert r["e_mixed_log"][g] == pytest.approx(-0.5, abs=1e-10)
            mult = _comb_brute(wt, oracle.comb_uniform(seed, 5 + g + 1))
            got = np.bincount(r["sources"][g], minlength=W)
            assert list(got) == mult
            mean = wt.mean()
            e_t = -0.5 - fb * math.log(mean)
            wt = np.full(W, mean)
        else:
            assert np.isnan(r["e_mixed_log"][g])
            assert list(r["sources"][g]) == list(range(W))
    assert n_branch == 4
    np.testing.assert_allclose(r["weights"], wt, rtol=1e-9)
    assert r["e_trial"] == pytest.approx(e_t, rel=1e-10)
    assert 0.5 < np.mean(r["bits"] & 1) <= 1.0


def test_run_clones_are_fresh_walkers_on_the_slot_streams():
    """After a reconfiguration slot j continues from the positions of walker source[j] on slot j's own random stream:
    redo the run with walkers rebuilt from positions alone (no clone) and compare decisions, positions and weights."""
    wl = qi.make_workload(0)
    osys = oracle.OracleSystem(wl.system)
    W, G, every, fb, tau, lim = 6, 4, 2, 1.0, 0.02, 1.0
    ids = [3, 4, 5, 6, 7, 8]
    start = wl.positions(0, W)
    r = oracle.dmc_run(osys, [osys.walker(p) for p in start], wl.seed, ids, 2, G, tau, lim, -17.0, every, fb)
    # by hand
    ws = [osys.walker(p) for p in start]
    e = [w.eloc()[0] for w in ws]
    wt = [1.0] * W
    e_t = -17.0
    some_copy = False
    for g in range(G):
        for n in range(W):
            b, e[n], wt[n], _ = ws[n].dmc_generation(wl.seed, ids[n], 2 + g, tau, lim, e_t, e[n], wt[n])
            assert np.array_equal(b & 1, r["bits"][g, :, n] & 1)
        if (g + 1) % every == 0:
            src = r["sources"][g]
            some_copy |= any(src[n] != n for n in range(W))
            em = sum(a * b for a, b in zip(wt, e)) / sum(wt)
            assert r["e_mixed_log"][g] == pytest.approx(em, rel=1e-12)
            pos = [ws[n].positions().copy() for n in range(W)]
            ws = [osys.walker(pos[src[n]]) for n in range(W)]
            e = [e[src[n]] for n in range(W)]
            mean = sum(wt) / W
            wt = [mean] * W
            e_t = em - fb * math.log(mean)
    assert some_copy
    for n in range(W):
        np.testing.assert_allclose(r["walkers"][n].positions(), ws[n].positions(), atol=1e-12)
        assert r["walkers"][n].eloc()[0] == pytest.approx(ws[n].eloc()[0], abs=1e-8)
    np.testing.assert_allclose(r["weights"], wt, rtol=1e-10)
    assert r["e_trial"] == pytest.approx(e_t, rel=1e-12)


def test_clone_is_independent_of_its_original():
    wl = qi.make_workload(0)
    osys = oracle.OracleSystem(wl.system)
    a = osys.walker(wl.positions(0, 1)[0])
    c = a.clone()
    ref = a.positions().copy()
    c.sweep(wl.seed, 0, 0, 0.05)
    assert np.array_equal(a.positions(), ref) and not np.array_equal(c.positions(), ref)
    b1 = a.sweep(wl.seed, 0, 0, 0.05)
    assert np.array_equal(a.positions(), c.positions())
    np.testing.assert_array_equal(a.Ainv(0), c.Ainv(0))
