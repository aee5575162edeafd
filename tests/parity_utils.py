"""Comparison protocol GPU vs oracle (BASELINE.json north_star tolerances).

The oracle side of a comparison does not depend on the GPU (both free-run from the same seeded positions), so it is
computed by `OracleFollower` threads -- one oracle walker each, advanced sweep by sweep in the background -- while the
GPU runs and while other tests run (`OracleFarm`, started by tests/conftest.py for the large configs).  Only a flagged
tie mismatch couples the two: the follower is then re-seeded from the GPU's positions and recomputes what follows."""
from __future__ import annotations

import threading

import numpy as np

import oracle
import paper_2504_07948_b200 as qb

TOL_RATIO = 1e-10      # ratios and log|Psi|, relative (ratios: for |rho_D e^dJ| >= RATIO_SMALL)
RATIO_SMALL = 1e-2     # below this the ratio is a cancelling dot product (proposal next to a node): its
TOL_RATIO_ABS = 1e-12  # rounding error is absolute, ~eps * sum_j |v_j x_j|, so it is held to this absolute bound
TOL_POS = 1e-10        # positions, absolute bohr (reading A27)
TOL_AINV = 1e-9        # A^-1, relative Frobenius
TOL_ELOC = 1e-9        # E_L, hartree


def rel_frob(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


FLOOR_FACTOR = 8       # GPU may be this many times further from the double oracle than that is from long double
RESYNC_EVERY = 10      # sweeps of free running between re-seeds of the oracle

_cpu_slots = threading.BoundedSemaphore(oracle.default_threads())   # oracle computations in flight, whoever asks


def cond2(ainv):
    """2-norm condition number of a Slater matrix from its (oracle) inverse."""
    sv = np.linalg.svd(ainv, compute_uv=False)
    return float(sv[0] / sv[-1])


class OracleFollower:
    """One oracle walker (double or long double), created and advanced sweep by sweep in a background thread.

    get(t) blocks until sweep t is done and returns its snapshot: bits, ratio, pacc [n_e], positions [n_e][3], logpsi,
    sign, eloc, ekin after the sweep.  creation() blocks until the walker exists and returns logpsi, sign, eloc, ekin
    (and cond(A) per spin if asked for) of the initial configuration.  reseed(t, pos) replaces the state after sweep t
    by a walker rebuilt from `pos` (comparison protocol); later sweeps are recomputed.  final_ainv(spin)
    is the inverse after the last sweep.  e_end limits every sweep to its first e_end electrons."""

    def __init__(self, osys, pos0, seed, walker_id, first_step, tau, n_sweeps, want_cond=False, e_end=None):
        self.osys, self.pos0, self.seed, self.wid = osys, np.array(pos0, np.float64), int(seed), int(walker_id)
        self.first_step, self.tau, self.n_sweeps, self.want_cond, self.e_end = int(first_step), float(tau), int(n_sweeps), want_cond, e_end
        self.cv = threading.Condition()
        self.snaps, self.epoch, self.pending, self._creation, self.error, self.walker = [], 0, None, None, None, None
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.thread.start()

    def _state(self, w):
        lp, sg = w.logpsi()
        e, k = w.eloc()
        return dict(positions=w.positions(), logpsi=lp, sign=sg, eloc=e, ekin=k)

    def _run(self):
        try:
            with _cpu_slots:
                w = self.osys.walker(self.pos0)
                c = self._state(w)
                if self.want_cond:
                    c["cond"] = [cond2(w.Ainv(sp)) if self.osys.ns(sp) else 1.0 for sp in (0, 1)]
            with self.cv:
                self.walker, self._creation = w, c
                self.cv.notify_all()
            while True:
                with self.cv:
                    while True:
                        if self.n_sweeps < 0:               # closed
                            return
                        if self.pending is not None or len(self.snaps) < self.n_sweeps:
                            break
                        self.cv.wait()                      # done; a late reseed wakes us up again
                    pend, self.pending = self.pending, None
                    t, ep = len(self.snaps), self.epoch
                with _cpu_slots:
                    if pend is not None:
                        w.set_positions(pend)
                    if t >= self.n_sweeps:
                        continue
                    ne = self.osys.n_elec
                    b, r, p = w.sweep_range(self.seed, self.wid, self.first_step + t, self.tau, 0, self.e_end or ne)
                    s = self._state(w)
                    s.update(bits=b, ratio=r, pacc=p)
                with self.cv:
                    if ep == self.epoch:
                        self.snaps.append(s)
                        self.cv.notify_all()
        except BaseException as e:  # noqa: BLE001 -- handed to the waiting test
            with self.cv:
                self.error = e
                self.cv.notify_all()

    def _wait(self, ready):
        with self.cv:
            while not ready() and self.error is None:
                self.cv.wait(1.0)
            if self.error is not None:
                raise self.error

    def creation(self):
        self._wait(lambda: self._creation is not None)
        return self._creation

    def get(self, t):
        assert t < self.n_sweeps
        self._wait(lambda: len(self.snaps) > t and self.pending is None)
        return self.snaps[t]

    def reseed(self, t, pos):
        with self.cv:
            del self.snaps[t + 1:]
            self.pending = np.array(pos, np.float64)
            self.epoch += 1
            self.cv.notify_all()

    def final_ainv(self, spin):
        self.get(self.n_sweeps - 1)
        return self.walker.Ainv(spin)

    def close(self):
        with self.cv:
            self.n_sweeps = -1
            self.cv.notify_all()


class OracleFarm:
    """Followers by (system, precision, walker, run parameters): asking twice returns the same follower, so a run can be
    started long before the test that compares it."""

    def __init__(self):
        self.systems, self.followers, self.lock = {}, {}, threading.Lock()

    def system(self, wl, long_double=False):
        key = (wl.config, wl.system.name, bool(long_double))
        with self.lock:
            if key not in self.systems:
                self.systems[key] = oracle.OracleSystem(wl.system, long_double=long_double)
            return self.systems[key]

    def request(self, wl, walker_ids, n_sweeps, first_step=0, long_double=False, want_cond=False, e_end=None):
        osys = self.system(wl, long_double)
        out = []
        for w in walker_ids:
            key = (wl.config, wl.system.name, bool(long_double), int(w), int(n_sweeps), int(first_step), wl.tau, e_end)
            with self.lock:
                if key not in self.followers:
                    self.followers[key] = OracleFollower(osys, wl.positions(w, w + 1)[0], wl.seed, w, first_step, wl.tau, n_sweeps,
                                                         want_cond=want_cond, e_end=e_end)
                out.append(self.followers[key])
        return out

    def close(self):
        for f in self.followers.values():
            f.close()
        self.followers.clear()
        self.systems.clear()


_FLOAT_KEYS = ("ratio_rel", "small_ratio_abs", "pos_abs", "logpsi_rel", "eloc_abs")


def _snap_distance(a_ratio, a_pos, a_logpsi, a_eloc, b):
    """deviations of (ratio, positions, logpsi, eloc) from snapshot b (the reference side)"""
    d = dict(ratio_rel=0.0, small_ratio_abs=0.0)
    m = np.abs(b["ratio"]) >= RATIO_SMALL
    if m.any():
        d["ratio_rel"] = float(np.max(np.abs(a_ratio[m] - b["ratio"][m]) / np.abs(b["ratio"][m])))
    if (~m).any():
        d["small_ratio_abs"] = float(np.max(np.abs(a_ratio[~m] - b["ratio"][~m])))
    d["pos_abs"] = float(np.abs(a_pos - b["positions"]).max())
    d["logpsi_rel"] = abs(a_logpsi - b["logpsi"]) / abs(b["logpsi"])
    d["eloc_abs"] = abs(a_eloc - b["eloc"])
    return d


def run_and_compare(wl, walker_ids, n_sweeps, delay_k, sweeps_per_call=1, threads=None, first_step=0, flags=qb.QMC_LOG_RATIOS,
                    gsys=None, osys=None, resync_every=RESYNC_EVERY, floor=False, crowd=None, floor_ids=None, floor_sweeps=None,
                    farm=None, want_cond=False, e_end=None, verbose=False):
    """Free-running comparison, walker by walker, sweep by sweep.

    The GPU runs the walkers `crowd` = (lo, hi) (default: exactly walker_ids, which must then be contiguous) as ONE crowd,
    the oracle follows the sampled walker_ids.  Returns a report dict; an unflagged accept/reject mismatch is recorded in
    rep["failures"].  A decision that differs with a tie flag on either side is flagged, not counted; the oracle walker is
    then re-seeded from the GPU positions and the comparison continues.

    Rounding differences between two correct FP64 evaluations grow along a trajectory (measured on config 0:
    1e-14 bohr after 1 sweep, 1e-11 after 100, and the long-double oracle drifts from the double oracle faster
    than the GPU does), so the floating-point tolerances are asserted on free-running windows of `resync_every`
    sweeps; at the end of a window every oracle walker is re-seeded from the GPU positions.  Accept/reject
    decisions are compared over the whole run.

    floor=True also runs the long-double build of the oracle on floor_ids (default: all sampled walkers) for the first
    floor_sweeps sweeps (default: all) and records how far the DOUBLE oracle is from it (floor_*; per sweep in
    rep["sweeps"]): two correct FP64 evaluations differ by ~cond(A) * 2^-53, so where that floor exceeds a BASELINE.json
    tolerance the test holds the GPU to FLOOR_FACTOR x the floor instead and says so (reading A26).

    e_end: compare only the first e_end electrons of every sweep (n_sweeps must then be 1: the state after a partial
    sweep is not the state the next sweep starts from)."""
    sysm = wl.system
    walker_ids = [int(w) for w in walker_ids]
    if crowd is None:
        crowd = (walker_ids[0], walker_ids[0] + len(walker_ids))
        assert walker_ids == list(range(*crowd))
    lo, hi = crowd
    assert all(lo <= w < hi for w in walker_ids) and (e_end is None or n_sweeps == 1)
    own_farm = farm is None
    farm = farm or OracleFarm()
    ow = farm.request(wl, walker_ids, n_sweeps, first_step, want_cond=want_cond, e_end=e_end)
    floor_ids = ([int(w) for w in floor_ids] if floor_ids is not None else walker_ids) if floor else []
    floor_sweeps = n_sweeps if floor_sweeps is None else min(floor_sweeps, n_sweeps)
    owl = dict(zip(floor_ids, farm.request(wl, floor_ids, floor_sweeps, first_step, long_double=True, e_end=e_end))) if floor else {}
    gsys = gsys or qb.qmc_init_from(sysm)
    gw = qb.qmc_walkers_create(gsys, wl.positions(lo, hi), wl.seed, first_walker_id=lo, first_step=first_step, flags=flags)
    rep = dict(n_moves=0, n_mismatch_flagged=0, n_resync=0, max_ratio_rel=0.0, max_small_ratio_abs=0.0, max_pos_abs=0.0, max_logpsi_rel=0.0,
               max_eloc_abs=0.0, max_ainv_rel=0.0, floor_ratio_rel=0.0, floor_small_ratio_abs=0.0, floor_pos_abs=0.0, floor_logpsi_rel=0.0,
               floor_eloc_abs=0.0, floor_ainv_rel=0.0, n_ties_gpu=0, n_ties_oracle=0, accept_frac=0.0, failures=[], sweeps=[],
               eloc_scale=0.0, walker_ids=walker_ids, floor_ids=floor_ids, floor_sweeps=floor_sweeps if floor else 0)
    ne = sysm.n_elec
    hi_e = e_end or ne
    acc = 0
    dead = set()   # walkers with an unflagged mismatch: reported once, not compared further
    for t in range(n_sweeps):
        qb.qmc_sweep(gw, 1, wl.tau, delay_k)
        gbits = qb.qmc_get_accept_log(gw).cpu().numpy()[0]          # [ne][W]
        gratio, gpacc = [x.cpu().numpy()[0] for x in qb.qmc_get_ratio_log(gw)]
        gpos = qb.qmc_get_positions(gw).cpu().numpy()
        glog, gsign = [x.cpu().numpy() for x in qb.qmc_get_logpsi(gw)]
        geloc, gekin = [x.cpu().numpy() for x in qb.qmc_get_eloc(gw)]
        row = dict(sweep=t, dev={k: 0.0 for k in _FLOAT_KEYS}, floor={k: 0.0 for k in _FLOAT_KEYS}, per_walker={})
        for n, w in enumerate(walker_ids):
            if w in dead:
                continue
            g = w - lo
            o = ow[n].get(t)
            gb, obits = gbits[:hi_e, g], o["bits"][:hi_e]
            rep["n_moves"] += len(gb)
            rep["n_ties_gpu"] += int(((gb & 2) != 0).sum())
            rep["n_ties_oracle"] += int(((obits & 2) != 0).sum())
            acc += int((gb & 1).sum())
            diff = np.nonzero((gb & 1) != (obits & 1))[0]
            if len(diff):
                i = int(diff[0])
                if (gb[i] & 2) or (obits[i] & 2):
                    rep["n_mismatch_flagged"] += 1
                    rep["n_resync"] += 1
                else:
                    rep["failures"].append(dict(walker=w, sweep=t, electron=i, gpu_pacc=float(gpacc[i, g]), oracle_pacc=float(o["pacc"][i]),
                                                gpu_ratio=float(gratio[i, g]), oracle_ratio=float(o["ratio"][i])))
                if e_end is not None:
                    dead.add(w)
                    continue
                ow[n].reseed(t, gpos[g])   # re-seed the oracle from the GPU state
                if w in owl and t < floor_sweeps:
                    owl[w].reseed(t, gpos[g])
                continue
            if e_end is None:
                d = _snap_distance(gratio[:, g], gpos[g], glog[g], geloc[g], o)
                assert int(gsign[g]) == o["sign"]
            else:  # a partial sweep: ratios only (the GPU's positions, log|Psi| and E_L are those after the whole sweep)
                oo = dict(o, ratio=o["ratio"][:hi_e], positions=np.zeros(3), logpsi=1.0, eloc=0.0)
                d = _snap_distance(gratio[:hi_e, g], np.zeros(3), 1.0, 0.0, oo)
            row["per_walker"][w] = dict(dev=d)
            for k in _FLOAT_KEYS:
                row["dev"][k] = max(row["dev"][k], d[k])
                rep["max_" + k] = max(rep["max_" + k], d[k])
            rep["eloc_scale"] = max(rep["eloc_scale"], abs(o["eloc"]))
            if w in owl and t < floor_sweeps:
                ol = owl[w].get(t)
                if np.array_equal(ol["bits"][:hi_e] & 1, obits & 1):
                    if e_end is None:
                        f = _snap_distance(o["ratio"], o["positions"], o["logpsi"], o["eloc"], ol)
                    else:
                        f = _snap_distance(o["ratio"][:hi_e], np.zeros(3), 1.0, 0.0, dict(ol, ratio=ol["ratio"][:hi_e], positions=np.zeros(3), logpsi=1.0, eloc=0.0))
                    row["per_walker"][w]["floor"] = f
                    for k in _FLOAT_KEYS:
                        row["floor"][k] = max(row["floor"][k], f[k])
                        rep["floor_" + k] = max(rep["floor_" + k], f[k])
                elif e_end is None:
                    owl[w].reseed(t, o["positions"])
        rep["sweeps"].append(row)
        if verbose:
            print(f"sweep {t}: dev " + " ".join(f"{k}={row['dev'][k]:.2e}" for k in _FLOAT_KEYS) +
                  (" | floor " + " ".join(f"{k}={row['floor'][k]:.2e}" for k in _FLOAT_KEYS) if floor and t < floor_sweeps else ""), flush=True)
        if resync_every and (t + 1) % resync_every == 0 and t + 1 < n_sweeps:
            for n, w in enumerate(walker_ids):
                ow[n].reseed(t, gpos[w - lo])
                if w in owl and t + 1 < floor_sweeps:
                    owl[w].reseed(t, gpos[w - lo])
    if e_end is None:
        rep["ainv_per_walker"] = {}
        for spin in (0, 1):
            if sysm.n_up == 0 if spin == 0 else sysm.n_dn == 0:
                continue
            ga = qb.qmc_get_Ainv(gw, spin).cpu().numpy()
            for n, w in enumerate(walker_ids):
                if w in dead:
                    continue
                oa = ow[n].final_ainv(spin)
                d = rel_frob(ga[w - lo], oa)
                rep["max_ainv_rel"] = max(rep["max_ainv_rel"], d)
                rep["ainv_per_walker"][(w, spin)] = dict(dev=d)
                if w in owl and floor_sweeps == n_sweeps:
                    f = rel_frob(oa, owl[w].final_ainv(spin))
                    rep["floor_ainv_rel"] = max(rep["floor_ainv_rel"], f)
                    rep["ainv_per_walker"][(w, spin)]["floor"] = f
    if want_cond:
        rep["cond"] = {w: ow[n].creation()["cond"] for n, w in enumerate(walker_ids)}
    rep["accept_frac"] = acc / max(rep["n_moves"], 1)
    rep["stats"] = qb.qmc_get_stats(gw)
    rep["n_gpu_walkers"] = hi - lo
    rep["gw"], rep["gsys"], rep["ow"], rep["osys"], rep["owl"] = gw, gsys, [f.walker for f in ow], farm.system(wl), owl
    if own_farm:
        for f in list(ow) + list(owl.values()):
            f.close()
    return rep
