"""Comparison protocol GPU vs oracle (BASELINE.json north_star tolerances).

The oracle side of a comparison does not depend on the GPU (both free-run from the same seeded positions), so it is
computed by `OracleFollower` threads -- one oracle walker each, advanced sweep by sweep in the background -- while the
GPU runs and while other tests run (`OracleFarm`, started by tests/conftest.py for the large configs).  Only a flagged
tie mismatch couples the two: the follower is then re-seeded from the GPU's positions and recomputes what follows."""
from __future__ import annotations

import os
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

# oracle computations in flight: one pool for the followers a test is waiting for, one for the background followers of the
# large configs (minutes per call, niced) -- which must not keep the foreground ones waiting for a slot
_fg_slots = threading.BoundedSemaphore(oracle.default_threads())
_bg_slots = threading.BoundedSemaphore(oracle.default_threads())


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

    def __init__(self, osys, pos0, seed, walker_id, first_step, tau, n_sweeps, want_cond=False, e_end=None, ld_inverse=False,
                 keep_ainv_at=(), carried_vs_fresh=False, background=False):
        self.osys, self.pos0, self.seed, self.wid = osys, np.array(pos0, np.float64), int(seed), int(walker_id)
        self.first_step, self.tau, self.n_sweeps, self.want_cond, self.e_end = int(first_step), float(tau), int(n_sweeps), want_cond, e_end
        self.ld_inverse, self.keep_ainv_at, self.carried_vs_fresh = ld_inverse, set(keep_ainv_at), carried_vs_fresh
        self.background = background   # started long before it is needed: yields the cores to whatever test is running now
        self.slots = _bg_slots if background else _fg_slots
        self.cv = threading.Condition()
        self.snaps, self.epoch, self.pending, self._creation, self.error, self.walker = [], 0, None, None, None, None
        self.horizon = self.n_sweeps   # sweeps the worker may compute ahead of the comparison (set_horizon)
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.thread.start()

    def _state(self, w):
        lp, sg = w.logpsi()
        e, k = w.eloc()
        return dict(positions=w.positions(), logpsi=lp, sign=sg, eloc=e, ekin=k)

    def _run(self):
        try:
            if self.background:
                try:
                    os.setpriority(os.PRIO_PROCESS, threading.get_native_id(), 10)   # Linux: per-thread nice value
                except (OSError, AttributeError):
                    pass
            with self.slots:
                w = self.osys.walker(self.pos0)
                if self.want_cond:
                    cond = [cond2(w.Ainv(sp)) if self.osys.ns(sp) else 1.0 for sp in (0, 1)]
                if self.ld_inverse:
                    # start from the LONG-DOUBLE LU inverse of the walker's own (double) Slater matrices, rounded to double:
                    # a second correct FP64 walker whose distance from the plain one is a conditioning floor (reading A26)
                    inv_floor = self._ld_inverse(w)
                c = self._state(w)
                if self.want_cond:
                    c["cond"] = cond
                if self.ld_inverse:
                    c["inv_floor"] = inv_floor
            with self.cv:
                self.walker, self._creation = w, c
                self.cv.notify_all()
            while True:
                with self.cv:
                    while True:
                        if self.n_sweeps < 0:               # closed
                            return
                        if self.pending is not None or len(self.snaps) < min(self.n_sweeps, self.horizon):
                            break
                        self.cv.wait()                      # done; a late reseed wakes us up again
                    pend, self.pending = self.pending, None
                    t, ep = len(self.snaps), self.epoch
                with self.slots:
                    if pend is not None:
                        w.set_positions(pend)
                        if self.ld_inverse:
                            self._ld_inverse(w)
                    if t >= self.n_sweeps:
                        continue
                    ne = self.osys.n_elec
                    b, r, p = w.sweep_range(self.seed, self.wid, self.first_step + t, self.tau, 0, self.e_end or ne)
                    s = self._state(w)
                    s.update(bits=b, ratio=r, pacc=p)
                    if t in self.keep_ainv_at or t == self.n_sweeps - 1:
                        s["ainv"] = [w.Ainv(sp) if self.osys.ns(sp) else None for sp in (0, 1)]
                    if self.carried_vs_fresh and t == self.n_sweeps - 1:
                        s["carried_vs_fresh"] = self._carried_vs_fresh(w, s)
                with self.cv:
                    if ep == self.epoch:
                        self.snaps.append(s)
                        self.cv.notify_all()
        except BaseException as e:  # noqa: BLE001 -- handed to the waiting test
            with self.cv:
                self.error = e
                self.cv.notify_all()

    def _ld_inverse(self, w):
        from concurrent.futures import ThreadPoolExecutor
        spins = [sp for sp in (0, 1) if self.osys.ns(sp)]

        def one(sp):
            rc, inv, _, _ = oracle.lu_inverse(w.A(sp), long_double=True)
            assert rc == 0
            return np.ascontiguousarray(inv.T)       # orientation of OracleWalker.Ainv()
        with ThreadPoolExecutor(max_workers=2) as ex:
            invs = list(ex.map(one, spins))
        floors = [0.0, 0.0]
        for sp, inv in zip(spins, invs):
            floors[sp] = rel_frob(w.Ainv(sp), inv)
            w.set_Ainv(sp, inv)
        return floors

    def _carried_vs_fresh(self, w, s):
        """the state carried through the sweeps against a walker built from scratch at the same positions"""
        f = self.osys.walker(s["positions"])
        lp, _ = f.logpsi()
        e, _ = f.eloc()
        return dict(ainv_rel=max(rel_frob(w.Ainv(sp), f.Ainv(sp)) for sp in (0, 1) if self.osys.ns(sp)),
                    logpsi_rel=abs(s["logpsi"] - lp) / abs(lp), eloc_abs=abs(s["eloc"] - e), eloc_scale=abs(e))

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

    def set_horizon(self, h):
        """do not compute beyond sweep h - 1 yet (what follows a re-seed would be thrown away)"""
        with self.cv:
            self.horizon = h
            self.cv.notify_all()

    def reseed(self, t, pos):
        with self.cv:
            del self.snaps[t + 1:]
            self.pending = np.array(pos, np.float64)
            self.epoch += 1
            self.cv.notify_all()

    def final_ainv(self, spin):
        return self.get(self.n_sweeps - 1)["ainv"][spin]

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

    def request(self, wl, walker_ids, n_sweeps, first_step=0, long_double=False, want_cond=False, e_end=None, ld_inverse=False,
                keep_ainv_at=(), carried_vs_fresh=False, positions=None, background=False):
        """positions (optional, [len(walker_ids)][n_e][3]): start from these instead of the workload's initial positions
        (a window that starts from the GPU's state); such followers are not shared."""
        osys = self.system(wl, long_double)
        out = []
        for n, w in enumerate(walker_ids):
            key = (wl.config, wl.system.name, bool(long_double), int(w), int(n_sweeps), int(first_step), wl.tau, e_end, bool(ld_inverse))
            with self.lock:
                if positions is not None:
                    key = key + (len(self.followers),)
                if key not in self.followers:
                    pos = positions[n] if positions is not None else wl.positions(w, w + 1)[0]
                    self.followers[key] = OracleFollower(osys, pos, wl.seed, w, first_step, wl.tau, n_sweeps, want_cond=want_cond, e_end=e_end,
                                                         ld_inverse=ld_inverse, keep_ainv_at=keep_ainv_at, carried_vs_fresh=carried_vs_fresh,
                                                         background=background)
                out.append(self.followers[key])
        return out

    def close(self):
        for f in self.followers.values():
            f.close()
        self.followers.clear()
        self.systems.clear()


_FLOAT_KEYS = ("ratio_rel", "small_ratio_abs", "pos_abs", "logpsi_rel", "eloc_abs")


def _snap_distance(a_ratio, a_pos, a_logpsi, a_eloc, b, hi_e=None):
    """deviations of (ratio, positions, logpsi, eloc) from snapshot b (the reference side); hi_e: only the first hi_e
    electrons of the sweep were run, so only their ratios mean anything"""
    d = dict(ratio_rel=0.0, small_ratio_abs=0.0, pos_abs=0.0, logpsi_rel=0.0, eloc_abs=0.0)
    br = b["ratio"][:hi_e]
    ar = a_ratio[:hi_e]
    m = np.abs(br) >= RATIO_SMALL
    if m.any():
        d["ratio_rel"] = float(np.max(np.abs(ar[m] - br[m]) / np.abs(br[m])))
    if (~m).any():
        d["small_ratio_abs"] = float(np.max(np.abs(ar[~m] - br[~m])))
    if hi_e is None:
        d["pos_abs"] = float(np.abs(a_pos - b["positions"]).max())
        d["logpsi_rel"] = abs(a_logpsi - b["logpsi"]) / abs(b["logpsi"])
        d["eloc_abs"] = abs(a_eloc - b["eloc"])
    return d


def run_and_compare(wl, walker_ids, n_sweeps, delay_k, first_step=0, flags=qb.QMC_LOG_RATIOS, gsys=None, resync_every=RESYNC_EVERY,
                    floor=False, crowd=None, floor_ids=None, floor_sweeps=None, farm=None, want_cond=False, e_end=None, verbose=False,
                    float_sweeps=None, ainv_at=None, gw=None, carried_vs_fresh=False):
    """Free-running comparison, walker by walker, sweep by sweep.

    The GPU runs the walkers `crowd` = (lo, hi) (default: exactly walker_ids, which must then be contiguous) as ONE crowd,
    the oracle follows the sampled walker_ids.  Returns a report dict; an unflagged accept/reject mismatch is recorded in
    rep["failures"].  A decision that differs with a tie flag on either side is flagged, not counted; the oracle walker is
    then re-seeded from the GPU positions and the comparison continues.

    Rounding differences between two correct FP64 evaluations grow along a trajectory -- it is the dynamics, not the
    kernels: the long-double oracle drifts from the double oracle as fast as the GPU does (measured
    on config 2: positions 1.5e-11 bohr apart after one sweep, 6e-6 after ten, decisions still identical) -- so the
    floating-point tolerances are asserted on free-running WINDOWS: the maxima rep["max_*"] cover the sweeps
    t < float_sweeps of the run (default: all), and at the end of every resync_every-th sweep all oracle walkers are
    re-seeded from the GPU positions.  Accept/reject decisions are compared over the whole run, and rep["sweeps"] records
    the deviations of every sweep.

    floor: how far two correct FP64 evaluations are apart here (reading A26).  True / "ld": the long-double build of the
    oracle runs floor_ids (default: all sampled walkers) for the first floor_sweeps sweeps (default: float_sweeps);
    rep["floor_*"] = distance of the DOUBLE oracle from it.  "ldinv": where a long-double sweep is out of reach, a second
    DOUBLE oracle walker starts from the long-double LU inverse of its own Slater matrices (OracleFollower ld_inverse);
    its distance from the plain double walker is a lower bound of the same floor.  Where the floor exceeds a
    BASELINE.json tolerance the tests hold the GPU to FLOOR_FACTOR x the floor instead and say so.

    gw: continue on existing GPU walkers (a window that starts from the GPU's state: the oracle walkers are built from
    the GPU's current positions, first_step must be the set's sweep counter).  ainv_at: sweeps after which A^-1 of the
    sampled walkers is compared (default: the last).  e_end: compare only the first e_end electrons of the (single) sweep."""
    sysm = wl.system
    walker_ids = [int(w) for w in walker_ids]
    if crowd is None:
        crowd = (walker_ids[0], walker_ids[0] + len(walker_ids))
        assert walker_ids == list(range(*crowd))
    lo, hi = crowd
    assert all(lo <= w < hi for w in walker_ids) and (e_end is None or n_sweeps == 1)
    float_sweeps = n_sweeps if float_sweeps is None else min(float_sweeps, n_sweeps)
    ainv_at = [n_sweeps - 1] if ainv_at is None else sorted(ainv_at)
    own_farm = farm is None
    farm = farm or OracleFarm()
    gsys = gsys or (gw.system if gw is not None else qb.qmc_init_from(sysm))
    start_pos = None
    if gw is None:
        gw = qb.qmc_walkers_create(gsys, wl.positions(lo, hi), wl.seed, first_walker_id=lo, first_step=first_step, flags=flags)
    else:
        assert gw.n_walkers == hi - lo
        start_pos = qb.qmc_get_positions(gw).cpu().numpy()
    pos_of = (lambda ids: None) if start_pos is None else (lambda ids: [start_pos[w - lo] for w in ids])
    ow = farm.request(wl, walker_ids, n_sweeps, first_step, want_cond=want_cond, e_end=e_end, keep_ainv_at=ainv_at,
                      carried_vs_fresh=carried_vs_fresh, positions=pos_of(walker_ids))
    if resync_every:
        for f in ow:
            f.set_horizon(resync_every)
    floor_mode = "ld" if floor is True else floor
    floor_ids = ([int(w) for w in floor_ids] if floor_ids is not None else walker_ids) if floor else []
    floor_sweeps = float_sweeps if floor_sweeps is None else min(floor_sweeps, n_sweeps)
    owl = {}
    if floor:
        fl = farm.request(wl, floor_ids, floor_sweeps, first_step, long_double=(floor_mode == "ld"), ld_inverse=(floor_mode == "ldinv"),
                          e_end=e_end, keep_ainv_at=[t for t in ainv_at if t < floor_sweeps], positions=pos_of(floor_ids))
        owl = dict(zip(floor_ids, fl))
    rep = dict(n_moves=0, n_mismatch_flagged=0, n_resync=0, max_ratio_rel=0.0, max_small_ratio_abs=0.0, max_pos_abs=0.0, max_logpsi_rel=0.0,
               max_eloc_abs=0.0, max_ainv_rel=0.0, floor_ratio_rel=0.0, floor_small_ratio_abs=0.0, floor_pos_abs=0.0, floor_logpsi_rel=0.0,
               floor_eloc_abs=0.0, floor_ainv_rel=0.0, n_ties_gpu=0, n_ties_oracle=0, accept_frac=0.0, failures=[], sweeps=[],
               eloc_scale=0.0, walker_ids=walker_ids, floor_ids=floor_ids, floor_sweeps=floor_sweeps if floor else 0, floor_mode=floor_mode,
               float_sweeps=float_sweeps, ainv_per_walker={})
    ne = sysm.n_elec
    hi_e = e_end or ne
    acc = 0
    dead = set()   # walkers whose oracle side stopped being comparable (mismatch in a partial sweep)
    st0 = qb.qmc_get_stats(gw)
    for t in range(n_sweeps):
        qb.qmc_sweep(gw, 1, wl.tau, delay_k)
        gbits = qb.qmc_get_accept_log(gw).cpu().numpy()[0]          # [ne][W]
        gratio, gpacc = [x.cpu().numpy()[0] for x in qb.qmc_get_ratio_log(gw)]
        gpos = qb.qmc_get_positions(gw).cpu().numpy()
        glog, gsign = [x.cpu().numpy() for x in qb.qmc_get_logpsi(gw)]
        geloc, gekin = [x.cpu().numpy() for x in qb.qmc_get_eloc(gw)]
        gainv = None
        if t in ainv_at and e_end is None:
            import torch
            idx = torch.tensor([w - lo for w in walker_ids], device="cuda")
            gainv = [qb.qmc_get_Ainv(gw, sp)[idx].cpu().numpy() if sysm_ns(sysm, sp) else None for sp in (0, 1)]
        row = dict(sweep=t, dev={k: 0.0 for k in _FLOAT_KEYS}, floor={k: 0.0 for k in _FLOAT_KEYS}, per_walker={})
        asserted = t < float_sweeps
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
            d = _snap_distance(gratio[:, g], gpos[g], glog[g], geloc[g], o, e_end)
            if e_end is None:
                assert int(gsign[g]) == o["sign"]
            pw = row["per_walker"][w] = dict(dev=d)
            for k in _FLOAT_KEYS:
                row["dev"][k] = max(row["dev"][k], d[k])
                if asserted:
                    rep["max_" + k] = max(rep["max_" + k], d[k])
            rep["eloc_scale"] = max(rep["eloc_scale"], abs(o["eloc"]))
            if gainv is not None:
                for sp in (0, 1):
                    if gainv[sp] is not None:
                        da = rel_frob(gainv[sp][n], o["ainv"][sp])
                        if asserted:
                            rep["max_ainv_rel"] = max(rep["max_ainv_rel"], da)
                        rep["ainv_per_walker"][(w, sp, t)] = dict(dev=da)
            if w in owl and t < floor_sweeps:
                ol = owl[w].get(t)
                if np.array_equal(ol["bits"][:hi_e] & 1, obits & 1):
                    f = _snap_distance(o["ratio"], o["positions"], o["logpsi"], o["eloc"], ol, e_end)
                    pw["floor"] = f
                    for k in _FLOAT_KEYS:
                        row["floor"][k] = max(row["floor"][k], f[k])
                        rep["floor_" + k] = max(rep["floor_" + k], f[k])
                    if gainv is not None and "ainv" in ol:
                        for sp in (0, 1):
                            if gainv[sp] is not None:
                                fa = rel_frob(o["ainv"][sp], ol["ainv"][sp])
                                rep["floor_ainv_rel"] = max(rep["floor_ainv_rel"], fa)
                                rep["ainv_per_walker"][(w, sp, t)]["floor"] = fa
                elif e_end is None:
                    owl[w].reseed(t, o["positions"])
        rep["sweeps"].append(row)
        if verbose:
            print(f"sweep {first_step + t}: dev " + " ".join(f"{k}={row['dev'][k]:.2e}" for k in _FLOAT_KEYS) +
                  (" | floor " + " ".join(f"{k}={row['floor'][k]:.2e}" for k in _FLOAT_KEYS) if floor and t < floor_sweeps else "") +
                  ("" if asserted else "   (free-running beyond the asserted window)"), flush=True)
        if resync_every and (t + 1) % resync_every == 0 and t + 1 < n_sweeps:
            for n, w in enumerate(walker_ids):
                ow[n].set_horizon(t + 1 + resync_every)
                ow[n].reseed(t, gpos[w - lo])
                if w in owl and t + 1 < floor_sweeps:
                    owl[w].reseed(t, gpos[w - lo])
    if want_cond:
        rep["cond"] = {w: ow[n].creation()["cond"] for n, w in enumerate(walker_ids)}
    if floor_mode == "ldinv":
        rep["inv_floor"] = {w: f.creation()["inv_floor"] for w, f in owl.items()}
    if carried_vs_fresh:
        rep["carried_vs_fresh"] = {w: ow[n].get(n_sweeps - 1)["carried_vs_fresh"] for n, w in enumerate(walker_ids) if w not in dead}
    rep["accept_frac"] = acc / max(rep["n_moves"], 1)
    st1 = qb.qmc_get_stats(gw)
    rep["stats"] = {k: st1[k] - (st0[k] if k != "nonfinite" else 0) for k in st1}
    rep["n_gpu_walkers"] = hi - lo
    rep["gw"], rep["gsys"], rep["ow"], rep["osys"], rep["owl"], rep["farm"] = gw, gsys, [f.walker for f in ow], farm.system(wl), owl, farm
    if own_farm:
        for f in list(ow) + list(owl.values()):
            f.close()
    return rep


REPORTS = []   # coverage / floor tables of the parity tests, printed by tests/conftest.py in the terminal summary


def note(text):
    REPORTS.append(text)
    print(text, flush=True)


def sysm_ns(sysm, spin):
    return sysm.n_up if spin == 0 else sysm.n_dn


def format_report(rep, title=""):
    """The table the tests print: per walker cond(A), raw deviation and measured floor (reading A26)."""
    lines = [f"--- {title}: {len(rep['walker_ids'])} sampled walkers of a crowd of {rep['n_gpu_walkers']}, {len(rep['sweeps'])} sweeps, "
             f"{rep['n_moves']} decisions compared, {len(rep['failures'])} unflagged mismatches, {rep['n_mismatch_flagged']} flagged; "
             f"floats asserted on the first {rep['float_sweeps']} sweep(s); floor: {rep['floor_mode'] or 'none'} on walkers {rep['floor_ids']}"]
    for row in rep["sweeps"]:
        lines.append(f"  sweep {row['sweep']}: dev " + " ".join(f"{k}={row['dev'][k]:.1e}" for k in _FLOAT_KEYS) +
                     (" | floor " + " ".join(f"{k}={row['floor'][k]:.1e}" for k in _FLOAT_KEYS) if row["sweep"] < rep["floor_sweeps"] else ""))
    if "cond" in rep:
        lines.append("  cond(A) [up, down] at creation: " + ", ".join(f"w{w}: {c[0]:.1e}/{c[1]:.1e}" for w, c in rep["cond"].items()))
    if "inv_floor" in rep:
        lines.append("  double vs long-double LU inverse (rel. Frobenius) [up, down]: " + ", ".join(f"w{w}: {c[0]:.1e}/{c[1]:.1e}" for w, c in rep["inv_floor"].items()))
    worst = sorted(rep["ainv_per_walker"].items(), key=lambda kv: -kv[1]["dev"])
    for (w, sp, t), v in worst[:6]:
        lines.append(f"  A^-1 walker {w} spin {sp} after sweep {t}: dev {v['dev']:.1e}" + (f" floor {v['floor']:.1e}" if "floor" in v else ""))
    if len(worst) > 6:
        lines.append(f"  ... {len(worst) - 6} more (walker, spin) inverses compared, every dev below {worst[6][1]['dev']:.1e}")
    lines.append("  maxima: " + " ".join(f"{k}={rep['max_' + k]:.1e}/{rep['floor_' + k]:.1e}" for k in _FLOAT_KEYS + ("ainv_rel",)) + "  (dev/floor)")
    return "\n".join(lines)


# ---------------------------------------------------------------------------------------- the large configs
# What the oracle follows at configs 1-3 (BASELINE.json configs; coverage stated in DESIGN.md section 6).  One place, so
# that tests/conftest.py can start exactly these followers when the GPU session starts and the tests find them running.
CFG1_IDS = list(range(0, 512, 16))            # 32 of the 512 walkers, 10 sweeps, long-double floor on all of them
CFG2_IDS = [0, 1, 37, 100, 127, 200, 254, 255]  # 8 of the 256 walkers
CFG2_FLOOR_IDS = [0, 100]                     # long-double oracle, first sweep (walker 100: cond(A) 5e6, the largest of the sample)
CFG2_FREE_SWEEPS = 9                          # free-running sweeps 0..8; sweep 9 is a second window started from the GPU's state
CFG3_IDS = [0, 21, 42, 63]                    # 4 of the 64 walkers, one whole sweep
CFG3_FLOOR_IDS = [42, 63]                     # walker 63: cond(A) 1.3e7
CFG4_EXTRA_IDS = [300, 511]                   # walkers beyond config 2's crowd (W = 512 points), first sweep


def request_large(farm, cfg):
    """Start (or find) the followers of one large config; returns the run_and_compare keyword arguments that use them."""
    import qmc_inputs as qi
    wl = qi.make_workload(cfg)
    if cfg == 1:
        kw = dict(walker_ids=CFG1_IDS, n_sweeps=10, crowd=(0, wl.n_walkers), floor="ld", want_cond=True, carried_vs_fresh=True)
    elif cfg == 2:
        kw = dict(walker_ids=CFG2_IDS, n_sweeps=CFG2_FREE_SWEEPS, crowd=(0, wl.n_walkers), floor="ld", floor_ids=CFG2_FLOOR_IDS, float_sweeps=1,
                  ainv_at=[0], want_cond=True, resync_every=0, carried_vs_fresh=True)
    elif cfg == 3:
        kw = dict(walker_ids=CFG3_IDS, n_sweeps=1, crowd=(0, wl.n_walkers), floor="ldinv", floor_ids=CFG3_FLOOR_IDS, want_cond=True,
                  carried_vs_fresh=True)
    else:
        raise ValueError(cfg)
    fs = kw.get("float_sweeps") or kw["n_sweeps"]
    ainv_at = kw.get("ainv_at") or [kw["n_sweeps"] - 1]
    bg = cfg in (2, 3)   # minutes of host time: started at session start, at low priority
    farm.request(wl, kw["walker_ids"], kw["n_sweeps"], want_cond=True, keep_ainv_at=ainv_at, carried_vs_fresh=kw.get("carried_vs_fresh", False),
                 background=bg)
    fl = kw.get("floor_ids") or kw["walker_ids"]
    farm.request(wl, fl, fs, long_double=(kw["floor"] == "ld"), ld_inverse=(kw["floor"] == "ldinv"), keep_ainv_at=[t for t in ainv_at if t < fs],
                 background=bg)
    if cfg == 2:
        farm.request(wl, CFG4_EXTRA_IDS, 1, background=True)
    return wl, kw
