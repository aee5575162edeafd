"""Several crowds per GPU (-m gpu): qmc_sweep_crowds advances walker sets of one system together on their own streams.
Each set must do exactly what qmc_sweep on it alone does, and match the oracle."""
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


def _state(gw):
    return (qb.qmc_get_accept_log(gw).cpu().numpy(), qb.qmc_get_positions(gw).cpu().numpy(), qb.qmc_get_eloc(gw)[0].cpu().numpy(),
            qb.qmc_get_logpsi(gw)[0].cpu().numpy(), qb.qmc_get_Ainv(gw, 0).cpu().numpy())


@pytest.mark.parametrize("cfg,sizes,T,k,flags,ctas", [(0, (24, 24), 3, 2, 2, 100), (0, (16, 9, 23), 2, 4, 2, 0), (0, (20, 20), 4, 1, 0, 0),
                                                      (1, (10, 10), 1, 32, 0, 120)])
def test_crowds_equal_the_sets_run_alone_and_the_oracle(cfg, sizes, T, k, flags, ctas):
    import torch
    wl = qi.make_workload(cfg)
    sysm = wl.system
    g = qb.qmc_init_from(sysm)
    firsts = np.concatenate([[0], np.cumsum(sizes)[:-1]])

    def make(stream_list):
        sets = []
        for c, (f, n) in enumerate(zip(firsts, sizes)):
            st = stream_list[c] if stream_list else None
            gw = qb.qmc_walkers_create(g, wl.positions(int(f), int(f + n)), wl.seed, first_walker_id=int(f), flags=flags, stream=st)
            if ctas:
                qb.qmc_set_mo_ctas(gw, ctas)
            sets.append(gw)
        return sets

    streams = [torch.cuda.Stream() for _ in sizes]
    together = make(streams)
    qb.qmc_sweep_crowds(together, T, wl.tau, k)
    alone = make(None)
    for gw in alone:
        qb.qmc_sweep(gw, T, wl.tau, k)
    torch.cuda.synchronize()
    osys = oracle.OracleSystem(sysm)
    for c, (a, b) in enumerate(zip(together, alone)):
        sa, sb = _state(a), _state(b)
        for x, y in zip(sa, sb):
            assert np.array_equal(x, y)                          # bit for bit: a set does not see the others
        assert qb.qmc_get_stats(a)["proposed"] == sizes[c] * sysm.n_elec * T
    # and the oracle, on the first walkers of the last crowd (global walker ids continue across crowds)
    bits, pos = _state(together[-1])[:2]
    for n in range(3):
        ow = osys.walker(wl.positions(int(firsts[-1]) + n, int(firsts[-1]) + n + 1)[0])
        ob = np.stack([ow.sweep(wl.seed, int(firsts[-1]) + n, t, wl.tau)[0] for t in range(T)])
        tie = ((bits[:, :, n] | ob) & 2) != 0
        assert np.array_equal((bits[:, :, n] & 1)[~tie], (ob & 1)[~tie])
        if not tie.any():
            assert np.abs(pos[n] - ow.positions()).max() < 1e-9


def test_crowds_argument_errors():
    wl = qi.make_workload(0)
    g = qb.qmc_init_from(wl.system)
    g2 = qb.qmc_init_from(wl.system)
    a = qb.qmc_walkers_create(g, wl.positions(0, 4), wl.seed)
    b = qb.qmc_walkers_create(g2, wl.positions(0, 4), wl.seed)
    with pytest.raises(qb.QmcError):
        qb.qmc_sweep_crowds([a, b], 1, wl.tau, 1)                 # two systems
    with pytest.raises(qb.QmcError):
        qb.qmc_sweep_crowds([a, a], 1, wl.tau, 1)                 # the same set twice
    with pytest.raises(qb.QmcError):
        qb.qmc_set_mo_ctas(a, 100000)
    qb.qmc_set_mo_ctas(a, 0)
    qb.qmc_sweep_crowds([a], 1, wl.tau, 1)
    assert qb.qmc_get_stats(a)["proposed"] == 4 * wl.system.n_elec


def test_stage_timers_and_contraction_residency_do_not_change_the_run():
    # the in-situ timers (qmc_set_profiling) bracket every n-th electron's launches with events and make the CTAs of the
    # sampled contractions stamp %globaltimer: the trajectory must not notice, every timed contraction has its stamps, and
    # a launch's mean CTA residency can never exceed its span (first CTA start to last CTA end)
    wl = qi.make_workload(1)
    g = qb.qmc_init_from(wl.system)
    runs = []
    for stride in (0, 4):
        gw = qb.qmc_walkers_create(g, wl.positions(0, 12), wl.seed, flags=qb.QMC_PER_ELECTRON)
        qb.qmc_set_profiling(gw, stride)
        qb.qmc_sweep(gw, 2, wl.tau, 16)
        runs.append(_state(gw))
        if stride:
            st = qb.qmc_get_stage_times(gw)
            span, span_min, residency, n = qb.qmc_get_mo_spans(gw)
            assert n == st["mo"][1] > 0
            assert st["mo"][0] > 0 and st["step"][1] > 0 and st["flush"][1] > 0
            assert 0 < residency <= span and 0 < span_min <= span
            assert qb.qmc_get_lanes(gw)[0] == 1
    for a, b in zip(*runs):
        assert np.array_equal(a, b)
