"""ctypes front end of the CPU oracle (oracle/qmc_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports
``paper_2504_07948_b200`` and shares no code with it.

The shared object is compiled on first use with the host's gcc (``-O3 -march=native``) into
``oracle/_build/``, keyed by source hash and CPU flags so that a build made on one machine is not
loaded on another.  ``build()`` is what ``__graft_entry__.build()`` calls.
"""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qmc_oracle.c")
_libs: dict = {}


def _cpu_tag() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return hashlib.sha1(line.encode()).hexdigest()[:8]
    except OSError:
        pass
    return "generic"


def build(long_double: bool = False) -> str:
    with open(_SRC, "rb") as f:
        h = hashlib.sha1(f.read()).hexdigest()[:10]
    out_dir = os.path.join(_HERE, "_build")
    os.makedirs(out_dir, exist_ok=True)
    name = f"liboracle_{'ld' if long_double else 'f64'}_{h}_{_cpu_tag()}.so"
    path = os.path.join(out_dir, name)
    if not os.path.exists(path):
        tmp = path + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O3", "-march=native", "-fPIC", "-shared", "-std=c11", "-o", tmp, _SRC, "-lm"]
        if long_double:
            cmd.insert(1, "-DORACLE_LONG_DOUBLE")
        subprocess.run(cmd, check=True, capture_output=True)
        os.replace(tmp, path)
    return path


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_u8p = C.POINTER(C.c_uint8)
_u32p = C.POINTER(C.c_uint32)


def _lib(long_double: bool = False):
    key = bool(long_double)
    if key in _libs:
        return _libs[key]
    lib = C.CDLL(build(long_double))
    lib.oracle_real_bytes.restype = C.c_int
    lib.oracle_system_create.restype = C.c_void_p
    lib.oracle_system_create.argtypes = [C.c_int, _dp, _dp, C.c_int, _ip, _ip, _ip, _ip, C.c_int, _dp, _dp,
                                         C.c_int, C.c_int, C.c_int, _dp, _dp, C.c_double, C.c_double,
                                         C.c_double, C.c_double]
    lib.oracle_system_destroy.argtypes = [C.c_void_p]
    lib.oracle_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
    lib.oracle_move_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _dp]
    lib.oracle_move_variates.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _dp, _dp]
    lib.oracle_basis_eval.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
    lib.oracle_mo_rows.argtypes = [C.c_void_p, C.c_int, _dp, _dp]
    lib.oracle_lu_inverse.restype = C.c_int
    lib.oracle_lu_inverse.argtypes = [C.c_int, _dp, _dp, _dp, _ip]
    lib.oracle_jastrow.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
    lib.oracle_walker_create.restype = C.c_void_p
    lib.oracle_walker_create.argtypes = [C.c_void_p, _dp]
    lib.oracle_walker_destroy.argtypes = [C.c_void_p]
    lib.oracle_walker_set_positions.restype = C.c_int
    lib.oracle_walker_set_positions.argtypes = [C.c_void_p, C.c_void_p, _dp]
    lib.oracle_walker_get_positions.argtypes = [C.c_void_p, _dp]
    lib.oracle_walker_get_Ainv.argtypes = [C.c_void_p, C.c_void_p, C.c_int, _dp]
    lib.oracle_walker_get_logpsi.argtypes = [C.c_void_p, _dp, _ip]
    lib.oracle_walker_get_A.argtypes = [C.c_void_p, C.c_void_p, C.c_int, _dp]
    lib.oracle_walker_set_Ainv.argtypes = [C.c_void_p, C.c_void_p, C.c_int, _dp]
    lib.oracle_walker_sweep.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_double,
                                        _u8p, _dp, _dp]
    lib.oracle_walker_sweep_range.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_double,
                                              C.c_int, C.c_int, _u8p, _dp, _dp]
    lib.oracle_walker_eloc.argtypes = [C.c_void_p, C.c_void_p, _dp, _dp]
    lib.oracle_walker_dmc_generation.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_double,
                                                 C.c_double, C.c_double, _dp, _dp, _dp, _u8p]
    lib.oracle_walker_sweep_limited.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_double,
                                                C.c_double, _u8p, _dp, _dp, _dp]
    lib.oracle_walker_clone.restype = C.c_void_p
    lib.oracle_walker_clone.argtypes = [C.c_void_p, C.c_void_p]
    lib.oracle_walker_deloc_dR.argtypes = [C.c_void_p, C.c_void_p, _dp]
    lib.oracle_walker_deloc_dR_atoms.argtypes = [C.c_void_p, C.c_void_p, C.c_int, _ip, _dp]
    lib.oracle_basis_eval_d3.argtypes = [C.c_void_p, _dp, _dp, _dp]
    lib.oracle_walker_vnl.restype = C.c_double
    lib.oracle_walker_vnl.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_int, _ip, _ip, _dp, _dp, _dp,
                                      C.c_int, _ip, _ip, _dp, _dp, _ip]
    lib.oracle_quadrature_directions.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _dp]
    lib.oracle_walker_dlogpsi_dR.argtypes = [C.c_void_p, C.c_void_p, _dp]
    lib.oracle_drift_limiter_scale.restype = C.c_double
    lib.oracle_drift_limiter_scale.argtypes = [C.c_double, C.c_double, C.c_double]
    lib.oracle_delayed_update.restype = C.c_int
    lib.oracle_delayed_update.argtypes = [C.c_int, _dp, C.c_int, _ip, _dp, _dp, _dp]
    lib.oracle_sherman_morrison.restype = C.c_double
    lib.oracle_sherman_morrison.argtypes = [C.c_int, _dp, C.c_int, _dp]
    lib.oracle_walker_logpsi_scratch.restype = C.c_int
    lib.oracle_walker_logpsi_scratch.argtypes = [C.c_void_p, C.c_void_p, _dp, _ip]
    _libs[key] = lib
    return lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


# ------------------------------------------------------------------ free functions

def philox4x32_10(ctr, key, long_double=False):
    c = np.asarray(ctr, np.uint32).copy()
    k = np.asarray(key, np.uint32).copy()
    o = np.zeros(4, np.uint32)
    _lib(long_double).oracle_philox4x32_10(c.ctypes.data_as(_u32p), k.ctypes.data_as(_u32p), o.ctypes.data_as(_u32p))
    return o


def move_uniforms(seed, walker, step, electron):
    U = np.zeros(5)
    _lib().oracle_move_uniforms(seed, walker, step, electron, _d(U))
    return U


def move_variates(seed, walker, step, electron, long_double=False):
    chi = np.zeros(3)
    u = C.c_double()
    _lib(long_double).oracle_move_variates(seed, walker, step, electron, _d(chi), C.byref(u))
    return chi, u.value


def lu_inverse(A, long_double=False):
    A = _f64(A)
    n = A.shape[0]
    Ainv = np.zeros_like(A)
    lad = C.c_double()
    sg = C.c_int()
    rc = _lib(long_double).oracle_lu_inverse(n, _d(A), _d(Ainv), C.byref(lad), C.byref(sg))
    return rc, Ainv, lad.value, sg.value


def sherman_morrison(Ainv, p, v, long_double=False):
    Ainv = _f64(Ainv).copy()
    v = _f64(v)
    rho = _lib(long_double).oracle_sherman_morrison(Ainv.shape[0], _d(Ainv), int(p), _d(v))
    return Ainv, rho


def delayed_update(A0inv, rows, Vrows, long_double=False):
    A0inv = _f64(A0inv)
    rows = _i32(rows)
    Vrows = _f64(Vrows)
    n, m = A0inv.shape[0], len(rows)
    out = np.zeros_like(A0inv)
    det = np.zeros(2)
    rc = _lib(long_double).oracle_delayed_update(n, _d(A0inv), m, rows.ctypes.data_as(_ip), _d(Vrows), _d(out), _d(det))
    return rc, out, det


# ------------------------------------------------------------------ system / walker handles

class OracleSystem:
    def __init__(self, system, long_double: bool = False):
        self.lib = _lib(long_double)
        self.long_double = long_double
        s = system
        self.n_basis, self.n_up, self.n_dn = s.n_basis, s.n_up, s.n_dn
        self.n_elec = s.n_up + s.n_dn
        self.n_atoms = s.n_atoms
        self._keep = [_f64(s.atoms_xyz), _f64(s.Z), _i32(s.shell_atom), _i32(s.shell_l), _i32(s.shell_nprim),
                      _i32(s.shell_prim_offset), _f64(s.alpha), _f64(s.coef), _f64(s.C_up), _f64(s.C_dn)]
        k = self._keep
        ip = lambda a: a.ctypes.data_as(_ip)
        self.h = self.lib.oracle_system_create(s.n_atoms, _d(k[0]), _d(k[1]), s.n_shells, ip(k[2]), ip(k[3]), ip(k[4]),
                                               ip(k[5]), len(k[6]), _d(k[6]), _d(k[7]), s.n_basis, s.n_up, s.n_dn,
                                               _d(k[8]), _d(k[9]), s.a_anti, s.a_para, s.b_ee, s.b_en)
        if not self.h:
            raise ValueError("oracle_system_create rejected the input")

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.oracle_system_destroy(self.h)
            self.h = None

    def ns(self, spin):
        return self.n_up if spin == 0 else self.n_dn

    def basis_eval(self, r):
        r = _f64(r)
        phi = np.zeros(self.n_basis)
        grad = np.zeros((3, self.n_basis))
        lap = np.zeros(self.n_basis)
        self.lib.oracle_basis_eval(self.h, _d(r), _d(phi), _d(grad), _d(lap))
        return phi, grad, lap

    def basis_eval_d3(self, r):
        """second derivatives [6][n_basis] (xx, yy, zz, xy, xz, yz) and gradient of the Laplacian [3][n_basis]"""
        r = _f64(r)
        hess = np.zeros((6, self.n_basis))
        glap = np.zeros((3, self.n_basis))
        self.lib.oracle_basis_eval_d3(self.h, _d(r), _d(hess), _d(glap))
        return hess, glap

    def mo_rows(self, spin, r):
        r = _f64(r)
        out = np.zeros((5, self.ns(spin)))
        self.lib.oracle_mo_rows(self.h, spin, _d(r), _d(out))
        return out

    def jastrow(self, R):
        R = _f64(R)
        J = C.c_double()
        grad = np.zeros((self.n_elec, 3))
        lap = np.zeros(self.n_elec)
        self.lib.oracle_jastrow(self.h, _d(R), C.byref(J), _d(grad), _d(lap))
        return J.value, grad, lap

    def walker(self, R):
        return OracleWalker(self, R)


class OracleWalker:
    def __init__(self, osys: OracleSystem, R):
        self.sys = osys
        self.lib = osys.lib
        R = _f64(R)
        assert R.shape == (osys.n_elec, 3)
        self.h = self.lib.oracle_walker_create(osys.h, _d(R))
        if not self.h:
            raise ArithmeticError("oracle: singular Slater matrix at walker creation")

    def __del__(self):
        if getattr(self, "h", None):
            self.lib.oracle_walker_destroy(self.h)
            self.h = None

    def sweep(self, seed, walker_id, step, tau):
        ne = self.sys.n_elec
        bits = np.zeros(ne, np.uint8)
        ratio = np.zeros(ne)
        pacc = np.zeros(ne)
        self.lib.oracle_walker_sweep(self.sys.h, self.h, seed, walker_id, step, tau, bits.ctypes.data_as(_u8p),
                                     _d(ratio), _d(pacc))
        return bits, ratio, pacc

    def sweep_range(self, seed, walker_id, step, tau, e_begin, e_end):
        """Electrons e_begin..e_end-1 of a sweep only (bounded sample for timing)."""
        ne = self.sys.n_elec
        bits = np.zeros(ne, np.uint8)
        ratio = np.zeros(ne)
        pacc = np.zeros(ne)
        self.lib.oracle_walker_sweep_range(self.sys.h, self.h, seed, walker_id, step, tau, int(e_begin), int(e_end),
                                           bits.ctypes.data_as(_u8p), _d(ratio), _d(pacc))
        return bits, ratio, pacc

    def clone(self):
        """Deep copy (what a DMC reconfiguration does to a walker that gets copies)."""
        c = object.__new__(OracleWalker)
        c.sys, c.lib = self.sys, self.lib
        c.h = self.lib.oracle_walker_clone(self.sys.h, self.h)
        return c

    def sweep_limited(self, seed, walker_id, step, tau, lim_a):
        """A sweep with the drift limiter of row f1; returns (bits, ratio, pacc, dr2[accepted, proposed])."""
        ne = self.sys.n_elec
        bits = np.zeros(ne, np.uint8)
        ratio = np.zeros(ne)
        pacc = np.zeros(ne)
        dr2 = np.zeros(2)
        self.lib.oracle_walker_sweep_limited(self.sys.h, self.h, seed, walker_id, step, tau, lim_a,
                                             bits.ctypes.data_as(_u8p), _d(ratio), _d(pacc), _d(dr2))
        return bits, ratio, pacc, dr2

    def dmc_generation(self, seed, walker_id, step, tau, lim_a, e_trial, e_old, weight):
        """One DMC generation (row f1): limited-drift sweep, E_L, tau_eff, weight update.
        Returns (bits, e_new, weight_new, tau_eff)."""
        bits = np.zeros(self.sys.n_elec, np.uint8)
        e = C.c_double(e_old)
        w = C.c_double(weight)
        te = C.c_double()
        self.lib.oracle_walker_dmc_generation(self.sys.h, self.h, seed, walker_id, step, tau, lim_a, e_trial,
                                              C.byref(e), C.byref(w), C.byref(te), bits.ctypes.data_as(_u8p))
        return bits, e.value, w.value, te.value

    def dlogpsi_dR(self):
        """d ln|Psi| / d R_a for every atom, [n_atoms][3] (row f2, first half; the paper's eq. 3 with lambda = R_a)."""
        out = np.zeros((self.sys.n_atoms, 3))
        self.lib.oracle_walker_dlogpsi_dR(self.sys.h, self.h, _d(out))
        return out

    def deloc_dR(self, atoms=None):
        """d E_L / d R_a for every atom (or the listed ones), [n][3] (row f2, second half; the paper's eq. 4)."""
        if atoms is not None:
            sel = np.ascontiguousarray(atoms, np.int32)
            out = np.zeros((len(sel), 3))
            self.lib.oracle_walker_deloc_dR_atoms(self.sys.h, self.h, len(sel), sel.ctypes.data_as(_ip), _d(out))
            return out
        out = np.zeros((self.sys.n_atoms, 3))
        self.lib.oracle_walker_deloc_dR(self.sys.h, self.h, _d(out))
        return out

    def vnl(self, ecp, seed, walker_id, step, details=False):
        """Non-local pseudopotential energy (row f3) with the quadrature rotations of (seed, walker_id, step).
        ecp: qmc_inputs.Ecp.  details=True: also (pair_i, pair_I, pts [n][12][3], ratios [n][12])."""
        ch_atom = np.ascontiguousarray(ecp.ch_atom, np.int32)
        ch_l = np.ascontiguousarray(ecp.ch_l, np.int32)
        beta, alpha, rcut = _f64(ecp.ch_beta), _f64(ecp.ch_alpha), _f64(ecp.rcut)
        assert rcut.shape == (self.sys.n_atoms,)
        cap = self.sys.n_elec * self.sys.n_atoms if details else 0
        pi, pI = np.zeros(max(cap, 1), np.int32), np.zeros(max(cap, 1), np.int32)
        pts, rat = np.zeros((max(cap, 1), 12, 3)), np.zeros((max(cap, 1), 12))
        n = C.c_int()
        v = self.lib.oracle_walker_vnl(self.sys.h, self.h, seed, walker_id, step, len(ch_l), ch_atom.ctypes.data_as(_ip),
                                       ch_l.ctypes.data_as(_ip), _d(beta), _d(alpha), _d(rcut), cap, pi.ctypes.data_as(_ip),
                                       pI.ctypes.data_as(_ip), _d(pts), _d(rat), C.byref(n))
        if details:
            k = n.value
            return v, pi[:k].copy(), pI[:k].copy(), pts[:k].copy(), rat[:k].copy()
        return v

    def eloc(self):
        e = C.c_double()
        k = C.c_double()
        self.lib.oracle_walker_eloc(self.sys.h, self.h, C.byref(e), C.byref(k))
        return e.value, k.value

    def positions(self):
        R = np.zeros((self.sys.n_elec, 3))
        self.lib.oracle_walker_get_positions(self.h, _d(R))
        return R

    def set_positions(self, R):
        R = _f64(R)
        rc = self.lib.oracle_walker_set_positions(self.sys.h, self.h, _d(R))
        if rc:
            raise ArithmeticError("oracle: singular Slater matrix")

    def Ainv(self, spin):
        n = self.sys.ns(spin)
        out = np.zeros((n, n))
        self.lib.oracle_walker_get_Ainv(self.sys.h, self.h, spin, _d(out))
        return out

    def A(self, spin):
        """the Slater matrix A[p][j] = phi_j(r_p) of one spin at the current positions (the cached value rows)"""
        n = self.sys.ns(spin)
        out = np.zeros((n, n))
        self.lib.oracle_walker_get_A(self.sys.h, self.h, spin, _d(out))
        return out

    def set_Ainv(self, spin, ainv):
        """replace the inverse of one spin (orientation of Ainv(): [p][j] = (A^-1)[j][p]); test use only (floors)"""
        a = _f64(ainv)
        assert a.shape == (self.sys.ns(spin),) * 2
        self.lib.oracle_walker_set_Ainv(self.sys.h, self.h, spin, _d(a))

    def logpsi(self):
        la = C.c_double()
        sg = C.c_int()
        self.lib.oracle_walker_get_logpsi(self.h, C.byref(la), C.byref(sg))
        return la.value, sg.value

    def logpsi_scratch(self):
        la = C.c_double()
        sg = C.c_int()
        rc = self.lib.oracle_walker_logpsi_scratch(self.sys.h, self.h, C.byref(la), C.byref(sg))
        if rc:
            raise ArithmeticError("oracle: singular Slater matrix")
        return la.value, sg.value


# ------------------------------------------------------------------ DMC reconfiguration (row f1, reading A30)

def drift_limiter_scale(v2, lim_a, tau, long_double=False):
    return _lib(long_double).oracle_drift_limiter_scale(float(v2), float(lim_a), float(tau))


def comb_uniform(seed, step):
    """The one uniform of a reconfiguration: Philox block 3 of counter (0xFFFFFFFF, step, 0xFFFFFFFF, 3), first word
    pair, mapped like every other uniform (A11)."""
    out = philox4x32_10([0xFFFFFFFF, step & 0xFFFFFFFF, 0xFFFFFFFF, 3], [seed & 0xFFFFFFFF, seed >> 32])
    x = (int(out[0]) << 32) | int(out[1])
    return (2 * (x >> 12) + 1) * 2.0 ** -53


def quadrature_directions(seed, walker_id, step, electron):
    """the 12 rotated icosahedron directions [12][3] of one (walker, step, electron)"""
    out = np.zeros((12, 3))
    _lib().oracle_quadrature_directions(seed, walker_id, step, electron, _d(out))
    return out


def comb_reconfigure(weights, xi):
    """Fixed-population "comb" reconfiguration, written out as its definition.

    W teeth at t_j = (j + xi) * (W_tot / W), j = 0..W-1, are laid over the cumulative weights c_i = w_0 + ... + w_i
    (summed in index order); walker i gets as many copies m_i as teeth fall in [c_{i-1}, c_i) (the last walker takes any
    tooth at or beyond c_{W-1}, which rounding can produce).  Walkers with m_i >= 1 stay in their slot; the k-th slot
    with m_i = 0 (ascending) receives the k-th extra copy, donors taken in ascending order, each m_i - 1 times.
    Returns (source, multiplicity, new_weight): slot j now holds a copy of old walker source[j]; every weight becomes
    W_tot / W."""
    w = np.asarray(weights, dtype=np.float64)
    W = len(w)
    tot = 0.0
    cum = np.zeros(W)
    for i in range(W):
        tot = tot + w[i]
        cum[i] = tot
    mult = np.zeros(W, dtype=np.int64)
    i = 0
    for j in range(W):
        t = (j + xi) * (tot / W)
        while i < W - 1 and not (t < cum[i]):
            i += 1
        mult[i] += 1
    source = np.arange(W, dtype=np.int64)
    dead = [k for k in range(W) if mult[k] == 0]
    extra = []
    for k in range(W):
        extra += [k] * max(0, int(mult[k]) - 1)
    assert len(dead) == len(extra)
    for d, e in zip(dead, extra):
        source[d] = e
    return source, mult, tot / W


def dmc_run(osys, walkers, seed, walker_ids, first_step, n_generations, tau, lim_a, e_trial0, branch_every, feedback,
            e_start=None, weights=None):
    """A DMC run with population control (row f1, reading A32), as the loop it is:
        for every generation g: every walker does dmc_generation with the current E_T;
        if branch_every > 0 and (g + 1) % branch_every == 0:
            e_mixed = sum w E_L / sum w; comb reconfiguration with the uniform of step first_step + g + 1 (walkers with
            copies are cloned into the dead slots, every weight becomes the mean weight);
            E_T <- e_mixed - feedback * ln(mean weight).
    Random streams belong to slots (walker_ids[slot]).  Returns a dict: walkers (list, after the run), bits
    [G][N_e][W], weights [W], eloc [W], e_trial_log [G] (the E_T in effect DURING generation g), e_mixed_log [G] (nan where
    no reconfiguration happened), sources [G][W] (slot map of each reconfiguration, identity elsewhere)."""
    W = len(walkers)
    walkers = list(walkers)
    e = np.array([w.eloc()[0] for w in walkers]) if e_start is None else np.array(e_start, float)
    wt = np.ones(W) if weights is None else np.array(weights, float)
    bits = np.zeros((n_generations, osys.n_elec, W), np.uint8)
    et_log, em_log = np.zeros(n_generations), np.full(n_generations, np.nan)
    sources = np.tile(np.arange(W), (n_generations, 1))
    e_t = float(e_trial0)
    for g in range(n_generations):
        et_log[g] = e_t
        for n in range(W):
            b, e[n], wt[n], _ = walkers[n].dmc_generation(seed, int(walker_ids[n]), first_step + g, tau, lim_a, e_t, e[n], wt[n])
            bits[g, :, n] = b
        if branch_every > 0 and (g + 1) % branch_every == 0:
            tot = 0.0
            ew = 0.0
            for n in range(W):
                tot = tot + wt[n]
                ew += wt[n] * e[n]
            em_log[g] = ew / tot
            src, mult, mean_w = comb_reconfigure(wt, comb_uniform(seed, first_step + g + 1))
            new_walkers = [walkers[n] if src[n] == n else walkers[src[n]].clone() for n in range(W)]
            walkers, e, wt = new_walkers, e[src].copy(), np.full(W, mean_w)
            sources[g] = src
            e_t = em_log[g] - feedback * np.log(mean_w)
    return dict(walkers=walkers, bits=bits, weights=wt, eloc=e, e_trial_log=et_log, e_mixed_log=em_log, sources=sources,
                e_trial=e_t)


# ------------------------------------------------------------------ crowd driver (threads over walkers)

def default_threads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return os.cpu_count() or 1


def run_crowd(system, positions, seed, walker_ids, first_step, n_sweeps, tau, threads=None, long_double=False,
              osys: OracleSystem | None = None):
    """Run independent walkers, parallel over walkers only (ctypes drops the GIL).

    Returns a dict: bits [T][N_e][W] uint8, ratio/pacc [T][N_e][W], eloc/ekin [T][W] (after each sweep),
    positions [W][N_e][3], logpsi [W], sign [W], walkers (list of OracleWalker, for getters)."""
    if osys is None:
        osys = OracleSystem(system, long_double)
    positions = _f64(positions)
    Wn = positions.shape[0]
    ne = osys.n_elec
    bits = np.zeros((n_sweeps, ne, Wn), np.uint8)
    ratio = np.zeros((n_sweeps, ne, Wn))
    pacc = np.zeros((n_sweeps, ne, Wn))
    eloc = np.zeros((n_sweeps, Wn))
    ekin = np.zeros((n_sweeps, Wn))
    walkers = [None] * Wn

    def one(n):
        w = osys.walker(positions[n])
        for t in range(n_sweeps):
            b, r, p = w.sweep(seed, int(walker_ids[n]), first_step + t, tau)
            bits[t, :, n], ratio[t, :, n], pacc[t, :, n] = b, r, p
            eloc[t, n], ekin[t, n] = w.eloc()
        walkers[n] = w

    nt = threads or default_threads()
    if nt <= 1 or Wn == 1:
        for n in range(Wn):
            one(n)
    else:
        with ThreadPoolExecutor(max_workers=nt) as ex:
            list(ex.map(one, range(Wn)))
    out_pos = np.stack([w.positions() for w in walkers])
    lp = np.array([w.logpsi() for w in walkers])
    return dict(bits=bits, ratio=ratio, pacc=pacc, eloc=eloc, ekin=ekin, positions=out_pos, logpsi=lp[:, 0],
                sign=lp[:, 1].astype(np.int8), walkers=walkers, osys=osys, threads=nt)
