"""Thin ctypes binding of the C ABI in include/qmc.h (same names, argument marshalling only).

PyTorch is used for device memory (output tensors) and streams; every step of the path runs in the
CUDA kernels of libqmc_b200.so.  There is no CPU fallback: if the library is missing or no sm_100
device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqmc_b200.so")

QMC_OK, QMC_ERR_ARG, QMC_ERR_CUDA, QMC_ERR_SINGULAR, QMC_ERR_NOMEM, QMC_ERR_STATE = 0, -1, -2, -3, -4, -5
QMC_LOG_RATIOS = 1
QMC_LARGE_PATH = 2
QMC_SCREEN_MO = 4
QMC_ONE_LANE = 8
QMC_PER_ELECTRON = 16
QMC_STEP_ONEPASS = 32
STAGES = ("step_half", "basis", "mo", "step", "flush", "eloc", "window")

EXPORTED = [
    "qmc_init", "qmc_finalize", "qmc_walkers_create", "qmc_walkers_destroy", "qmc_sweep", "qmc_get_positions",
    "qmc_get_Ainv", "qmc_get_logpsi", "qmc_get_eloc", "qmc_get_accept_log", "qmc_get_ratio_log", "qmc_get_stats",
    "qmc_synchronize", "qmc_eval_basis", "qmc_eval_basis_noalloc", "qmc_eval_mo", "qmc_time_stage", "qmc_set_profiling", "qmc_get_stage_times",
    "qmc_measure_fp64_peak", "qmc_launch_count", "qmc_last_error", "qmc_version",
    "qmc_dmc_step", "qmc_get_weights", "qmc_branch", "qmc_get_mo_work", "qmc_get_dlogpsi_dR",
    "qmc_dmc_run", "qmc_get_deloc_dR", "qmc_set_ecp", "qmc_get_vnl", "qmc_set_mo_ctas", "qmc_sweep_crowds",
    "qmc_release_scratch", "qmc_philox_words", "qmc_get_lanes", "qmc_get_mo_spans", "qmc_stale_error",
]


class QmcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"qmc error {code}: {msg}")
        self.code = code


class _Atoms(C.Structure):
    _fields_ = [("n_atoms", C.c_int), ("xyz", C.c_void_p), ("Z", C.c_void_p)]


class _Basis(C.Structure):
    _fields_ = [("n_shells", C.c_int), ("atom", C.c_void_p), ("l", C.c_void_p), ("n_prim", C.c_void_p),
                ("prim_offset", C.c_void_p), ("n_prim_total", C.c_int), ("alpha", C.c_void_p), ("coef", C.c_void_p)]


class _Mo(C.Structure):
    _fields_ = [("n_basis", C.c_int), ("n_up", C.c_int), ("n_dn", C.c_int), ("C_up", C.c_void_p), ("C_dn", C.c_void_p)]


class _Jastrow(C.Structure):
    _fields_ = [("a_anti", C.c_double), ("a_para", C.c_double), ("b_ee", C.c_double), ("b_en", C.c_double)]


_lib = None


def load_library(path: str | None = None):
    """Load libqmc_b200.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise QmcError(QMC_ERR_STATE, f"{p} not found: build it with `python -m paper_2504_07948_b200.build` "
                                      "(there is no CPU fallback)")
    lib = C.CDLL(p)
    vp, i, d, u64, u32 = C.c_void_p, C.c_int, C.c_double, C.c_uint64, C.c_uint32
    lib.qmc_init.argtypes = [C.POINTER(vp), C.POINTER(_Atoms), C.POINTER(_Basis), C.POINTER(_Mo), C.POINTER(_Jastrow), vp]
    lib.qmc_finalize.argtypes = [vp]
    lib.qmc_finalize.restype = None
    lib.qmc_walkers_create.argtypes = [vp, C.POINTER(vp), i, vp, u64, u32, u32, u32, vp]
    lib.qmc_walkers_destroy.argtypes = [vp]
    lib.qmc_walkers_destroy.restype = None
    lib.qmc_sweep.argtypes = [vp, i, d, i]
    lib.qmc_get_positions.argtypes = [vp, vp]
    lib.qmc_get_Ainv.argtypes = [vp, i, vp]
    lib.qmc_get_logpsi.argtypes = [vp, vp, vp]
    lib.qmc_get_eloc.argtypes = [vp, vp, vp]
    lib.qmc_get_accept_log.argtypes = [vp, vp]
    lib.qmc_get_ratio_log.argtypes = [vp, vp, vp]
    lib.qmc_get_stats.argtypes = [vp] + [C.POINTER(u64)] * 4
    lib.qmc_synchronize.argtypes = [vp]
    lib.qmc_eval_basis.argtypes = [vp, i, vp, vp, vp]
    lib.qmc_eval_basis_noalloc.argtypes = [vp, i, vp, vp, vp]
    lib.qmc_eval_mo.argtypes = [vp, i, i, vp, vp, vp]
    lib.qmc_time_stage.argtypes = [vp, i, i, i, i, C.POINTER(d)]
    lib.qmc_set_profiling.argtypes = [vp, i]
    lib.qmc_get_stage_times.argtypes = [vp, C.POINTER(d), C.POINTER(u64)]
    lib.qmc_measure_fp64_peak.argtypes = [d, C.POINTER(d), vp]
    lib.qmc_dmc_step.argtypes = [vp, i, d, i, d, d]
    lib.qmc_get_weights.argtypes = [vp, vp, vp]
    lib.qmc_branch.argtypes = [vp, vp, C.POINTER(d)]
    lib.qmc_get_dlogpsi_dR.argtypes = [vp, vp]
    lib.qmc_get_deloc_dR.argtypes = [vp, vp, vp]
    lib.qmc_set_ecp.argtypes = [vp, i, vp, vp, vp, vp, vp]
    lib.qmc_get_vnl.argtypes = [vp, vp, C.POINTER(u64)]
    lib.qmc_set_mo_ctas.argtypes = [vp, i]
    lib.qmc_sweep_crowds.argtypes = [C.POINTER(vp), i, i, d, i]
    lib.qmc_dmc_run.argtypes = [vp, i, d, i, d, d, i, d, C.POINTER(d), vp, vp]
    lib.qmc_get_mo_work.argtypes = [vp, C.POINTER(u64), C.POINTER(u64)]
    lib.qmc_release_scratch.argtypes = [vp]
    lib.qmc_get_lanes.argtypes = [vp, C.POINTER(i), C.POINTER(i)]
    lib.qmc_get_mo_spans.argtypes = [vp, C.POINTER(d), C.POINTER(d), C.POINTER(d), C.POINTER(u64)]
    lib.qmc_philox_words.argtypes = [i, vp, vp, vp]
    lib.qmc_launch_count.restype = u64
    lib.qmc_last_error.restype = C.c_char_p
    lib.qmc_stale_error.restype = C.c_char_p
    lib.qmc_version.restype = C.c_char_p
    for name in EXPORTED:
        fn = getattr(lib, name)
        if name not in ("qmc_finalize", "qmc_walkers_destroy", "qmc_launch_count", "qmc_last_error", "qmc_version", "qmc_stale_error"):
            fn.restype = i
    if path is None:
        _lib = lib
    return lib


def _check(rc):
    if rc != 0:
        raise QmcError(rc, load_library().qmc_last_error().decode())


def _stream_ptr(stream=None):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _ptr(x):
    """Raw pointer of a numpy array (host) or a torch tensor (host or device)."""
    if x is None:
        return C.c_void_p(0)
    if isinstance(x, np.ndarray):
        return C.c_void_p(x.ctypes.data)
    return C.c_void_p(x.data_ptr())


# ------------------------------------------------------------------ the ABI, same names

class System:
    """Handle returned by qmc_init."""

    def __init__(self, handle, n_basis, n_up, n_dn, stream):
        self.handle, self.n_basis, self.n_up, self.n_dn, self.stream = handle, n_basis, n_up, n_dn, stream
        self.n_elec = n_up + n_dn

    def ns(self, spin):
        return self.n_up if spin == 0 else self.n_dn

    def close(self):
        if self.handle:
            load_library().qmc_finalize(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Walkers:
    """Handle returned by qmc_walkers_create."""

    def __init__(self, handle, system, n_walkers, stream, flags):
        self.handle, self.system, self.n_walkers, self.stream, self.flags = handle, system, n_walkers, stream, flags
        self.last_nsteps = 0   # `stream`: the torch stream all work of this set is enqueued on

    def close(self):
        if self.handle:
            load_library().qmc_walkers_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def qmc_init(atoms_xyz, Z, shell_atom, shell_l, shell_nprim, shell_prim_offset, alpha, coef, n_basis, n_up, n_dn,
             C_up, C_dn, a_anti=0.5, a_para=0.25, b_ee=1.0, b_en=1.0, stream=None) -> System:
    """qmc_init(atoms, basis, mo_coeffs, jastrow).  Array arguments: numpy (host) or torch (host/device)."""
    lib = load_library()
    f64 = lambda a: np.ascontiguousarray(a, np.float64) if isinstance(a, (np.ndarray, list, tuple)) else a
    i32 = lambda a: np.ascontiguousarray(a, np.int32) if isinstance(a, (np.ndarray, list, tuple)) else a
    keep = [f64(atoms_xyz), f64(Z), i32(shell_atom), i32(shell_l), i32(shell_nprim), i32(shell_prim_offset),
            f64(alpha), f64(coef), f64(C_up), f64(C_dn) if C_dn is not None else None]
    at = _Atoms(len(keep[1]), _ptr(keep[0]), _ptr(keep[1]))
    ba = _Basis(len(keep[3]), _ptr(keep[2]), _ptr(keep[3]), _ptr(keep[4]), _ptr(keep[5]), len(keep[6]), _ptr(keep[6]), _ptr(keep[7]))
    mo = _Mo(n_basis, n_up, n_dn, _ptr(keep[8]), _ptr(keep[9]) if n_dn > 0 else C.c_void_p(0))
    ja = _Jastrow(a_anti, a_para, b_ee, b_en)
    h = C.c_void_p()
    sp = _stream_ptr(stream)
    _check(lib.qmc_init(C.byref(h), C.byref(at), C.byref(ba), C.byref(mo), C.byref(ja), sp))
    sysh = System(h, n_basis, n_up, n_dn, stream)
    sysh.n_atoms = len(keep[1])
    return sysh


def qmc_init_from(system, stream=None) -> System:
    """Convenience: qmc_init from a qmc_inputs.System-like object (attribute marshalling only)."""
    s = system
    return qmc_init(s.atoms_xyz, s.Z, s.shell_atom, s.shell_l, s.shell_nprim, s.shell_prim_offset, s.alpha, s.coef,
                    s.n_basis, s.n_up, s.n_dn, s.C_up, s.C_dn, s.a_anti, s.a_para, s.b_ee, s.b_en, stream)


def qmc_finalize(system: System):
    system.close()


def qmc_walkers_create(system: System, positions, seed, first_walker_id=0, first_step=0, flags=0, stream=None) -> Walkers:
    lib = load_library()
    if isinstance(positions, (list, tuple)):
        positions = np.asarray(positions, np.float64)
    if isinstance(positions, np.ndarray):
        positions = np.ascontiguousarray(positions, np.float64)
        shape = positions.shape
    else:
        positions = positions.contiguous()
        shape = tuple(positions.shape)
    if len(shape) != 3 or shape[1] != system.n_elec or shape[2] != 3:
        raise QmcError(QMC_ERR_ARG, f"positions must be [W][{system.n_elec}][3], got {shape}")
    h = C.c_void_p()
    import torch
    stream = stream if stream is not None else torch.cuda.current_stream()
    _check(lib.qmc_walkers_create(system.handle, C.byref(h), shape[0], _ptr(positions), C.c_uint64(seed),
                                  first_walker_id, first_step, flags, _stream_ptr(stream)))
    return Walkers(h, system, shape[0], stream, flags)


def qmc_walkers_destroy(walkers: Walkers):
    walkers.close()


def qmc_sweep(walkers: Walkers, nsteps, tau, delay_k):
    _check(load_library().qmc_sweep(walkers.handle, int(nsteps), float(tau), int(delay_k)))
    walkers.last_nsteps = int(nsteps)


def qmc_sweep_crowds(sets, nsteps, tau, delay_k):
    """qmc_sweep of several walker sets of one system together (electron by electron, each set on its own stream)."""
    arr = (C.c_void_p * len(sets))(*[w.handle for w in sets])
    _check(load_library().qmc_sweep_crowds(arr, len(sets), int(nsteps), float(tau), int(delay_k)))
    for w in sets:
        w.last_nsteps = int(nsteps)


def qmc_dmc_step(walkers: Walkers, n_generations, tau, delay_k, e_trial, limiter_a=1.0):
    _check(load_library().qmc_dmc_step(walkers.handle, int(n_generations), float(tau), int(delay_k), float(e_trial), float(limiter_a)))
    walkers.last_nsteps = int(n_generations)


def qmc_get_weights(walkers: Walkers, out=None, out_tau_eff=None):
    import torch
    out = _out((walkers.n_walkers,), torch.float64, out)
    out_tau_eff = _out((walkers.n_walkers,), torch.float64, out_tau_eff)
    with _ordered(walkers, out, out_tau_eff):
        _check(load_library().qmc_get_weights(walkers.handle, _ptr(out), _ptr(out_tau_eff)))
    return out, out_tau_eff


def qmc_get_dlogpsi_dR(walkers: Walkers, out=None):
    """d ln|Psi| / d R_a, [W][n_atoms][3] (row f2, first half)."""
    import torch
    out = _out((walkers.n_walkers, walkers.system.n_atoms, 3), torch.float64, out)
    with _ordered(walkers, out):
        _check(load_library().qmc_get_dlogpsi_dR(walkers.handle, _ptr(out)))
    return out


def qmc_get_deloc_dR(walkers: Walkers, out=None, out_dlogpsi=None, with_dlogpsi=True):
    """(d E_L / d R_a, d ln|Psi| / d R_a), each [W][n_atoms][3] (row f2; eqs. 3 and 4); the second is None if not asked for."""
    import torch
    shape = (walkers.n_walkers, walkers.system.n_atoms, 3)
    out = _out(shape, torch.float64, out)
    if with_dlogpsi:
        out_dlogpsi = _out(shape, torch.float64, out_dlogpsi)
    with _ordered(walkers, out, out_dlogpsi):
        _check(load_library().qmc_get_deloc_dR(walkers.handle, _ptr(out), _ptr(out_dlogpsi) if with_dlogpsi else None))
    return out, (out_dlogpsi if with_dlogpsi else None)


def qmc_set_ecp(system: System, ecp):
    """Attach the non-local pseudopotential channels (qmc_inputs.Ecp) to a system (row f3)."""
    import numpy as np
    ch_atom = np.ascontiguousarray(ecp.ch_atom, np.int32)
    ch_l = np.ascontiguousarray(ecp.ch_l, np.int32)
    beta = np.ascontiguousarray(ecp.ch_beta, np.float64)
    alpha = np.ascontiguousarray(ecp.ch_alpha, np.float64)
    rcut = np.ascontiguousarray(ecp.rcut, np.float64)
    _check(load_library().qmc_set_ecp(system.handle, len(ch_l), ch_atom.ctypes.data, ch_l.ctypes.data, beta.ctypes.data,
                                      alpha.ctypes.data, rcut.ctypes.data))


def qmc_get_vnl(walkers: Walkers, out=None):
    """(V_nl [W] tensor, number of (electron, atom) pairs inside the cut-offs) at the current configuration (row f3)."""
    import torch
    out = _out((walkers.n_walkers,), torch.float64, out)
    n = C.c_uint64()
    with _ordered(walkers, out):
        _check(load_library().qmc_get_vnl(walkers.handle, _ptr(out), C.byref(n)))
    return out, n.value


def qmc_release_scratch(walkers: Walkers):
    """Free the scratch kept by the row-f2 / f3 getters and the host-pointer getters."""
    _check(load_library().qmc_release_scratch(walkers.handle))


def qmc_philox_words(ctr_key, stream=None):
    """Raw Philox4x32-10 words of the move kernels' generator: ctr_key [n][6] uint32 (counter 0..3, key 0..1) -> [n][4]."""
    ck = np.ascontiguousarray(ctr_key, np.uint32)
    assert ck.ndim == 2 and ck.shape[1] == 6
    out = np.zeros((ck.shape[0], 4), np.uint32)
    _check(load_library().qmc_philox_words(ck.shape[0], _ptr(ck), _ptr(out), _stream_ptr(stream)))
    return out


def qmc_get_lanes(walkers: Walkers):
    """(n_lanes, [walkers of lane 0, walkers of lane 1])"""
    n = C.c_int()
    per = (C.c_int * 2)()
    _check(load_library().qmc_get_lanes(walkers.handle, C.byref(n), per))
    return n.value, [per[0], per[1]]


def qmc_get_mo_spans(walkers: Walkers):
    """(mean span, min span, mean CTA residency) in microseconds of the profiled contraction launches on the GPU, and how
    many were recorded"""
    a, b, c, n = C.c_double(), C.c_double(), C.c_double(), C.c_uint64()
    _check(load_library().qmc_get_mo_spans(walkers.handle, C.byref(a), C.byref(b), C.byref(c), C.byref(n)))
    return a.value, b.value, c.value, n.value


def qmc_set_mo_ctas(walkers: Walkers, n_ctas):
    """Grid of this walker set's MO contraction (0 = all SMs); smaller leaves SMs to crowds on other streams."""
    _check(load_library().qmc_set_mo_ctas(walkers.handle, int(n_ctas)))


def qmc_get_mo_work(walkers: Walkers):
    """(executed, dense) (tile, k-block) iterations of the MO contraction since creation (QMC_SCREEN_MO sets only)."""
    a, b = C.c_uint64(), C.c_uint64()
    _check(load_library().qmc_get_mo_work(walkers.handle, C.byref(a), C.byref(b)))
    return a.value, b.value


def qmc_branch(walkers: Walkers, out_source=None):
    """Comb reconfiguration; returns (source [W] int32 tensor, e_mixed float)."""
    import torch
    out_source = _out((walkers.n_walkers,), torch.int32, out_source)
    e = C.c_double()
    with _ordered(walkers, out_source):
        _check(load_library().qmc_branch(walkers.handle, _ptr(out_source), C.byref(e)))
    return out_source, e.value


def qmc_dmc_run(walkers: Walkers, n_generations, tau, delay_k, e_trial0, limiter_a=1.0, branch_every=1, feedback=1.0):
    """DMC run with population control on the device; returns (e_trial after the run, branch_log [n_branch][3] float64
    tensor = {e_mixed, E_T after, W_tot / W}, sources [n_branch][W] int32 tensor)."""
    import torch
    nb = int(n_generations) // int(branch_every) if branch_every > 0 else 0
    log = torch.empty((nb, 3), dtype=torch.float64, device="cuda")
    src = torch.empty((nb, walkers.n_walkers), dtype=torch.int32, device="cuda")
    e = C.c_double()
    with _ordered(walkers, log, src):
        _check(load_library().qmc_dmc_run(walkers.handle, int(n_generations), float(tau), int(delay_k), float(e_trial0), float(limiter_a),
                                          int(branch_every), float(feedback), C.byref(e), _ptr(log) if nb else None, _ptr(src) if nb else None))
    walkers.last_nsteps = int(n_generations)
    return e.value, log, src


def _out(shape, dtype, out, device="cuda"):
    import torch
    if out is not None:
        return out
    return torch.empty(shape, dtype=dtype, device=device)


class _ordered:
    """Stream ordering of a getter (ordering contract of include/qmc.h): the library writes device outputs
    asynchronously on the WALKER SET's stream, while the caller's tensors live on torch's current stream.  When the two
    differ, the set's stream first waits for the current one (a freshly allocated output may be a recycled block still in
    use there), and after the call the current stream waits for the set's, and the caching allocator is told the tensors
    are in use on that stream.  Same stream: nothing to do."""

    def __init__(self, walkers, *tensors):
        import torch
        self.ws, self.cur, self.tensors = walkers.stream, torch.cuda.current_stream(), tensors
        self.cross = self.ws is not None and self.ws.cuda_stream != self.cur.cuda_stream

    def __enter__(self):
        if self.cross:
            self.ws.wait_stream(self.cur)
        return self

    def __exit__(self, *exc):
        if self.cross:
            self.cur.wait_stream(self.ws)
            for t in self.tensors:
                if t is not None and hasattr(t, "is_cuda") and t.is_cuda:
                    t.record_stream(self.ws)
        return False


def qmc_get_positions(walkers: Walkers, out=None):
    import torch
    out = _out((walkers.n_walkers, walkers.system.n_elec, 3), torch.float64, out)
    with _ordered(walkers, out):
        _check(load_library().qmc_get_positions(walkers.handle, _ptr(out)))
    return out


def qmc_get_Ainv(walkers: Walkers, spin, out=None):
    import torch
    n = walkers.system.ns(spin)
    out = _out((walkers.n_walkers, n, n), torch.float64, out)
    with _ordered(walkers, out):
        _check(load_library().qmc_get_Ainv(walkers.handle, int(spin), _ptr(out)))
    return out


def qmc_get_logpsi(walkers: Walkers, out=None, out_sign=None):
    import torch
    out = _out((walkers.n_walkers,), torch.float64, out)
    out_sign = _out((walkers.n_walkers,), torch.int8, out_sign)
    with _ordered(walkers, out, out_sign):
        _check(load_library().qmc_get_logpsi(walkers.handle, _ptr(out), _ptr(out_sign)))
    return out, out_sign


def qmc_get_eloc(walkers: Walkers, out=None, out_kin=None):
    import torch
    out = _out((walkers.n_walkers,), torch.float64, out)
    out_kin = _out((walkers.n_walkers,), torch.float64, out_kin)
    with _ordered(walkers, out, out_kin):
        _check(load_library().qmc_get_eloc(walkers.handle, _ptr(out), _ptr(out_kin)))
    return out, out_kin


def qmc_get_accept_log(walkers: Walkers, out=None):
    import torch
    out = _out((walkers.last_nsteps, walkers.system.n_elec, walkers.n_walkers), torch.uint8, out)
    if out.numel():
        with _ordered(walkers, out):
            _check(load_library().qmc_get_accept_log(walkers.handle, _ptr(out)))
    return out


def qmc_get_ratio_log(walkers: Walkers, out=None, out_pacc=None):
    import torch
    shape = (walkers.last_nsteps, walkers.system.n_elec, walkers.n_walkers)
    out = _out(shape, torch.float64, out)
    out_pacc = _out(shape, torch.float64, out_pacc)
    with _ordered(walkers, out, out_pacc):
        _check(load_library().qmc_get_ratio_log(walkers.handle, _ptr(out), _ptr(out_pacc)))
    return out, out_pacc


def qmc_get_stats(walkers: Walkers):
    v = [C.c_uint64() for _ in range(4)]
    _check(load_library().qmc_get_stats(walkers.handle, *[C.byref(x) for x in v]))
    return dict(zip(("proposed", "accepted", "ties", "nonfinite"), [x.value for x in v]))


def qmc_synchronize(walkers: Walkers):
    _check(load_library().qmc_synchronize(walkers.handle))


def qmc_eval_basis(system: System, xyz, out=None, stream=None):
    import torch
    n = int(xyz.shape[0])
    if isinstance(xyz, np.ndarray):
        xyz = np.ascontiguousarray(xyz, np.float64)
    out = _out((n, 5, system.n_basis), torch.float64, out)
    _check(load_library().qmc_eval_basis(system.handle, n, _ptr(xyz), _ptr(out), _stream_ptr(stream)))
    return out


def qmc_eval_basis_noalloc(system: System, xyz, out, stream=None):
    """qmc_eval_basis without any device allocation (include/qmc.h): `xyz` [n][3] and `out` [n][5][n_basis] are the caller's
    CUDA float64 tensors; the call only enqueues on the stream and does not synchronise."""
    import torch
    for t, name in ((xyz, "xyz"), (out, "out")):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise TypeError(f"qmc_eval_basis_noalloc: {name} must be a contiguous CUDA float64 tensor")
    n = int(xyz.shape[0])
    if tuple(xyz.shape) != (n, 3) or tuple(out.shape) != (n, 5, system.n_basis):
        raise ValueError("qmc_eval_basis_noalloc: xyz must be [n][3] and out [n][5][n_basis]")
    _check(load_library().qmc_eval_basis_noalloc(system.handle, n, _ptr(xyz), _ptr(out), _stream_ptr(stream)))
    return out


def qmc_eval_mo(system: System, spin, xyz, out=None, stream=None):
    import torch
    n = int(xyz.shape[0])
    if isinstance(xyz, np.ndarray):
        xyz = np.ascontiguousarray(xyz, np.float64)
    out = _out((n, 5, system.ns(spin)), torch.float64, out)
    _check(load_library().qmc_eval_mo(system.handle, int(spin), n, _ptr(xyz), _ptr(out), _stream_ptr(stream)))
    return out


def qmc_time_stage(walkers: Walkers, stage, spin=0, delay_k=1, reps=10) -> float:
    if isinstance(stage, str):
        stage = STAGES.index(stage)
    ms = C.c_double()
    _check(load_library().qmc_time_stage(walkers.handle, stage, spin, delay_k, reps, C.byref(ms)))
    return ms.value


def qmc_set_profiling(walkers: Walkers, stride):
    _check(load_library().qmc_set_profiling(walkers.handle, int(stride)))


def qmc_get_stage_times(walkers: Walkers):
    ms = (C.c_double * 7)()
    n = (C.c_uint64 * 7)()
    _check(load_library().qmc_get_stage_times(walkers.handle, ms, n))
    return {STAGES[i]: (ms[i], n[i]) for i in range(7)}


def qmc_measure_fp64_peak(ms_target=200.0, stream=None) -> float:
    t = C.c_double()
    _check(load_library().qmc_measure_fp64_peak(float(ms_target), C.byref(t), _stream_ptr(stream)))
    return t.value


def qmc_launch_count() -> int:
    return int(load_library().qmc_launch_count())


def qmc_version() -> str:
    return load_library().qmc_version().decode()


def qmc_stale_error() -> str:
    return load_library().qmc_stale_error().decode()


def qmc_last_error() -> str:
    return load_library().qmc_last_error().decode()
