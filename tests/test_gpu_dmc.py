"""Row f1 (DMC generation) on the GPU against the oracle, through the C ABI (-m gpu): accept/reject decisions of the
limited-drift sweeps identical, tau_eff and weights to 1e-10 relative, E_L to 1e-9 Ha, the comb's slot map identical
when both sides see the same weights, and the copied walkers carry their whole state (they keep matching the oracle
for further generations)."""
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


def _oracle_generations(osys, walkers, seed, ids, step0, T, tau, a, e_t, e_old, weight):
    """T generations of every oracle walker; returns bits [T][ne][W], e [W], weight [W], tau_eff [W] (last)."""
    W = len(walkers)
    bits = np.zeros((T, osys.n_elec, W), np.uint8)
    e_old, weight = np.array(e_old, float), np.array(weight, float)
    te = np.zeros(W)
    for n, w in enumerate(walkers):
        for t in range(T):
            b, e_old[n], weight[n], te[n] = w.dmc_generation(seed, int(ids[n]), step0 + t, tau, a, e_t, e_old[n], weight[n])
            bits[t, :, n] = b
    return bits, e_old, weight, te


def _compare(gw, bits_o, e_o, w_o, te_o, eloc_tol=1e-9):
    bits = qb.qmc_get_accept_log(gw).cpu().numpy()
    wts, te = (x.cpu().numpy() for x in qb.qmc_get_weights(gw))
    eloc = qb.qmc_get_eloc(gw)[0].cpu().numpy()
    diff = (bits & 1) != (bits_o & 1)
    assert not np.any(diff & (((bits | bits_o) & 2) == 0)), "unflagged accept/reject mismatch"
    ok = ~np.any(diff, axis=(0, 1))                    # walkers without a (flagged) tie mismatch
    assert ok.sum() >= len(ok) - 1
    np.testing.assert_allclose(te[ok], te_o[ok], rtol=1e-12)
    np.testing.assert_allclose(wts[ok], w_o[ok], rtol=1e-10)
    assert np.abs(eloc[ok] - e_o[ok]).max() < eloc_tol
    return ok


@pytest.mark.parametrize("cfg,W,k,T,e_t,flags", [(0, 48, 1, 12, -76.0, 0), (0, 48, 1, 12, -76.0, 2), (0, 48, 4, 12, -76.0, 2),
                                                 (1, 12, 32, 2, -550.0, 0)])
def test_dmc_generations_match_oracle(cfg, W, k, T, e_t, flags):
    # flags 0: config 0 takes the one-launch small-system path (row f4); 2 = QMC_LARGE_PATH: the per-electron kernels
    wl = qi.make_workload(cfg)
    sysm = wl.system
    a, tau = 1.0, wl.tau
    pos = wl.positions(0, W)
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, wl.seed, flags=flags)
    e0 = qb.qmc_get_eloc(gw)[0].cpu().numpy()
    qb.qmc_dmc_step(gw, T, tau, k, e_t, a)
    osys = oracle.OracleSystem(sysm)
    ows = [osys.walker(pos[n]) for n in range(W)]
    e_start = np.array([w.eloc()[0] for w in ows])
    assert np.abs(e_start - e0).max() < 1e-9
    bits_o, e_o, w_o, te_o = _oracle_generations(osys, ows, wl.seed, range(W), 0, T, tau, a, e_t, e_start, np.ones(W))
    ok = _compare(gw, bits_o, e_o, w_o, te_o, eloc_tol=1e-9 if cfg == 0 else 1e-7)
    assert ok.all() or cfg == 0
    st = qb.qmc_get_stats(gw)
    assert st["proposed"] == W * sysm.n_elec * T and st["nonfinite"] == 0
    wts = qb.qmc_get_weights(gw)[0].cpu().numpy()
    assert np.all(wts > 0) and np.std(wts) > 0          # the weights actually moved


def test_limiter_changes_trajectories_and_zero_switches_it_off():
    wl = qi.make_workload(0)
    pos = wl.positions(0, 16)
    g = qb.qmc_init_from(wl.system)
    runs = {}
    for a in (0.0, 1.0):
        gw = qb.qmc_walkers_create(g, pos, wl.seed)
        qb.qmc_dmc_step(gw, 3, wl.tau, 1, -76.0, a)
        runs[a] = (qb.qmc_get_accept_log(gw).cpu().numpy(), qb.qmc_get_positions(gw).cpu().numpy())
    gw = qb.qmc_walkers_create(g, pos, wl.seed)
    qb.qmc_sweep(gw, 3, wl.tau, 1)
    plain = (qb.qmc_get_accept_log(gw).cpu().numpy(), qb.qmc_get_positions(gw).cpu().numpy())
    assert np.array_equal(runs[0.0][0], plain[0]) and np.array_equal(runs[0.0][1], plain[1])   # a = 0 is reading A6
    assert np.abs(runs[1.0][1] - plain[1]).max() > 1e-4                                          # a = 1 is not


def test_hydrogen_weights_closed_form_on_gpu():
    sysm = qi.hydrogen_atom()
    g = qb.qmc_init_from(sysm)
    rng = np.random.default_rng(2)
    W, T, tau, e_t = 32, 25, 0.05, -0.45
    pos = rng.standard_normal((W, 1, 3))
    gw = qb.qmc_walkers_create(g, pos, 123)
    qb.qmc_dmc_step(gw, T, tau, 1, e_t, 1.0)
    bits = qb.qmc_get_accept_log(gw).cpu().numpy()            # [T][1][W]
    wts, te = (x.cpu().numpy() for x in qb.qmc_get_weights(gw))
    n_acc = (bits[:, 0, :] & 1).sum(axis=0).astype(np.float64)
    # one electron: tau_eff is tau on an accepted move and 0 otherwise; E_L = -1/2 exactly
    np.testing.assert_allclose(wts, np.exp(-n_acc * tau * (-0.5 - e_t)), rtol=1e-10)
    assert np.all((te == 0.0) | (np.abs(te - tau) < 1e-15))
    assert np.abs(qb.qmc_get_eloc(gw)[0].cpu().numpy() + 0.5).max() < 1e-10


def test_branch_slot_map_copies_and_continuation():
    wl = qi.make_workload(0)
    sysm = wl.system
    W, k, a, tau, e_t = 40, 2, 1.0, wl.tau, -75.0          # e_t off the mean energy: weights spread quickly
    pos = wl.positions(0, W)
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, wl.seed)
    qb.qmc_dmc_step(gw, 8, 4 * tau, k, e_t, a)
    w_before = qb.qmc_get_weights(gw)[0].cpu().numpy()
    pos_before = qb.qmc_get_positions(gw).cpu().numpy()
    eloc_before = qb.qmc_get_eloc(gw)[0].cpu().numpy()
    ainv_before = qb.qmc_get_Ainv(gw, 0).cpu().numpy()
    src_t, e_mixed = qb.qmc_branch(gw)
    src = src_t.cpu().numpy()
    # the oracle's comb on the same weights, same uniform (Philox counter (0xFFFFFFFF, step = 8, 0xFFFFFFFF, 3))
    src_o, mult_o, w_new = oracle.comb_reconfigure(w_before, oracle.comb_uniform(wl.seed, 8))
    assert np.array_equal(src, src_o)
    assert (mult_o == 0).sum() >= 1, "test needs at least one copy"
    assert e_mixed == pytest.approx(float((w_before * eloc_before).sum() / w_before.sum()), rel=1e-12)
    wts = qb.qmc_get_weights(gw)[0].cpu().numpy()
    assert np.all(wts == w_new)
    # every slot holds exactly the state of its source
    assert np.array_equal(qb.qmc_get_positions(gw).cpu().numpy(), pos_before[src])
    assert np.array_equal(qb.qmc_get_eloc(gw)[0].cpu().numpy(), eloc_before[src])
    assert np.array_equal(qb.qmc_get_Ainv(gw, 0).cpu().numpy(), ainv_before[src])
    # and keeps evolving like an oracle walker started from that state under the SLOT's random stream
    T2 = 3
    qb.qmc_dmc_step(gw, T2, tau, k, e_t, a)
    osys = oracle.OracleSystem(sysm)
    ows = [osys.walker(pos_before[src[n]]) for n in range(W)]
    bits_o, e_o, w_o, te_o = _oracle_generations(osys, ows, wl.seed, range(W), 8, T2, tau, a, e_t, eloc_before[src],
                                                 np.full(W, w_new))
    _compare(gw, bits_o, e_o, w_o, te_o, eloc_tol=1e-8)
    copies = np.nonzero(src != np.arange(W))[0]
    pos_after = qb.qmc_get_positions(gw).cpu().numpy()
    for d in copies:                                            # a copy and its donor have diverged (different streams)
        assert np.abs(pos_after[d] - pos_after[src[d]]).max() > 1e-6


# ------------------------------------------------------------------ qmc_dmc_run: the loop with population control

def test_hydrogen_run_closed_form_on_gpu():
    sysm = qi.hydrogen_atom()
    g = qb.qmc_init_from(sysm)
    rng = np.random.default_rng(4)
    W, G, every, fb, tau, seed, e_t0 = 64, 20, 4, 0.5, 0.08, 99, -0.4
    gw = qb.qmc_walkers_create(g, rng.standard_normal((W, 1, 3)), seed)
    e_t_end, log, src = qb.qmc_dmc_run(gw, G, tau, 1, e_t0, 1.0, every, fb)
    log, src = log.cpu().numpy(), src.cpu().numpy()
    bits = qb.qmc_get_accept_log(gw).cpu().numpy()            # [G][1][W]
    assert bits.shape == (G, 1, W) and log.shape == (G // every, 3)
    wt, e_t, nb = np.ones(W), e_t0, 0
    for gen in range(G):
        wt = wt * np.exp(tau * (bits[gen, 0] & 1) * (0.5 + e_t))
        if (gen + 1) % every == 0:
            assert log[nb, 0] == pytest.approx(-0.5, abs=1e-10)
            s_o, _, mean = oracle.comb_reconfigure(wt, oracle.comb_uniform(seed, gen + 1))
            assert np.array_equal(src[nb], s_o)
            e_t = -0.5 - fb * math.log(mean)
            assert log[nb, 1] == pytest.approx(e_t, rel=1e-10) and log[nb, 2] == pytest.approx(mean, rel=1e-10)
            wt = np.full(W, mean)
            nb += 1
    assert e_t_end == pytest.approx(e_t, rel=1e-10)
    np.testing.assert_allclose(qb.qmc_get_weights(gw)[0].cpu().numpy(), wt, rtol=1e-9)


@pytest.mark.parametrize("flags,k,every", [(0, 1, 2), (2, 1, 2), (2, 4, 3), (0, 1, 0)])
def test_dmc_run_matches_the_oracle_loop(flags, k, every):
    wl = qi.make_workload(0)
    sysm = wl.system
    W, G, fb, tau, lim, e_t0 = 24, 6, 1.0, 3 * wl.tau, 1.0, -75.0
    pos = wl.positions(0, W)
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, pos, wl.seed, flags=flags)
    e_t_end, log, src = qb.qmc_dmc_run(gw, G, tau, k, e_t0, lim, every, fb)
    log, src = log.cpu().numpy(), src.cpu().numpy()
    osys = oracle.OracleSystem(sysm)
    r = oracle.dmc_run(osys, [osys.walker(p) for p in pos], wl.seed, range(W), 0, G, tau, lim, e_t0, every, fb)
    bits = qb.qmc_get_accept_log(gw).cpu().numpy()
    diff = (bits & 1) != (r["bits"] & 1)
    assert not np.any(diff), "accept/reject mismatch (a flagged tie would also end the comparison of a branching run)"
    gens = [gi for gi in range(G) if every > 0 and (gi + 1) % every == 0]
    assert len(gens) == log.shape[0] == src.shape[0]
    for nb, gi in enumerate(gens):
        assert np.array_equal(src[nb], r["sources"][gi])
        assert log[nb, 0] == pytest.approx(r["e_mixed_log"][gi], abs=1e-8)
        assert log[nb, 1] == pytest.approx(r["e_trial_log"][gi + 1] if gi + 1 < G else r["e_trial"], abs=1e-8)
    if every:
        assert any(np.any(s != np.arange(W)) for s in src), "test needs at least one copy"
    assert e_t_end == pytest.approx(r["e_trial"], abs=1e-8)
    np.testing.assert_allclose(qb.qmc_get_weights(gw)[0].cpu().numpy(), r["weights"], rtol=1e-9)
    assert np.abs(qb.qmc_get_eloc(gw)[0].cpu().numpy() - r["eloc"]).max() < 1e-8
    po = np.stack([w.positions() for w in r["walkers"]])
    assert np.abs(qb.qmc_get_positions(gw).cpu().numpy() - po).max() < 1e-9
    st = qb.qmc_get_stats(gw)
    assert st["proposed"] == W * sysm.n_elec * G


def test_dmc_run_equals_the_calls_it_replaces():
    """qmc_dmc_run is qmc_dmc_step + qmc_branch + the E_T rule, minus the host round trips: bit for bit."""
    wl = qi.make_workload(0)
    W, G, every, fb, tau = 32, 6, 2, 0.7, 2 * wl.tau
    pos = wl.positions(0, W)
    g = qb.qmc_init_from(wl.system)
    a = qb.qmc_walkers_create(g, pos, wl.seed, flags=2)
    e_end, log, src = qb.qmc_dmc_run(a, G, tau, 3, -76.0, 1.0, every, fb)
    b = qb.qmc_walkers_create(g, pos, wl.seed, flags=2)
    e_t = -76.0
    for gi in range(G):
        qb.qmc_dmc_step(b, 1, tau, 3, e_t, 1.0)
        if (gi + 1) % every == 0:
            s, em = qb.qmc_branch(b)
            mean = float(qb.qmc_get_weights(b)[0][0])
            e_t = em - fb * math.log(mean)
            assert np.array_equal(s.cpu().numpy(), src[(gi + 1) // every - 1].cpu().numpy())
    assert e_end == pytest.approx(e_t, rel=1e-14)
    assert np.array_equal(qb.qmc_get_positions(a).cpu().numpy(), qb.qmc_get_positions(b).cpu().numpy())
    np.testing.assert_allclose(qb.qmc_get_weights(a)[0].cpu().numpy(), qb.qmc_get_weights(b)[0].cpu().numpy(), rtol=1e-13)


def test_config2_full_size_generation_sampled():
    """Row f1 at the size and in the launch configuration bench.py times (256-water config, 256 walkers, delay 64):
    one DMC generation of the whole crowd, two sampled walkers against the oracle's generation."""
    from concurrent.futures import ThreadPoolExecutor
    wl = qi.make_workload(2)
    sysm = wl.system
    g = qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(g, wl.positions(), wl.seed)
    e0 = qb.qmc_get_eloc(gw)[0].cpu().numpy()
    e_t = float(e0.mean())
    qb.qmc_dmc_step(gw, 1, wl.tau, wl.delay_k, e_t, 1.0)
    bits = qb.qmc_get_accept_log(gw).cpu().numpy()
    wts, te = (x.cpu().numpy() for x in qb.qmc_get_weights(gw))
    el = qb.qmc_get_eloc(gw)[0].cpu().numpy()
    osys = oracle.OracleSystem(sysm)

    def one(n):
        ow = osys.walker(wl.positions(n, n + 1)[0])
        e_start = ow.eloc()[0]
        return (n, e_start) + tuple(ow.dmc_generation(wl.seed, n, 0, wl.tau, 1.0, e_t, e_start, 1.0))
    with ThreadPoolExecutor(max_workers=2) as ex:
        res = list(ex.map(one, [3, 254]))
    for n, e_start, ob, e_new, w_new, te_o in res:
        assert abs(e0[n] - e_start) < 1e-6
        d = (bits[0, :, n] & 1) != (ob & 1)
        assert not np.any(d & (((bits[0, :, n] | ob) & 2) == 0)), "unflagged accept/reject mismatch"
        if not d.any():
            assert te[n] == pytest.approx(te_o, rel=1e-12)
            assert abs(el[n] - e_new) < 1e-6                      # reading A26: 1e-9 relative to the energy scale
            # the exponent tau_eff (E_old + E_new)/2 carries the absolute error of E_L
            assert wts[n] == pytest.approx(w_new, rel=1e-8)
