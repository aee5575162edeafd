"""Seeded synthetic inputs for the batched Slater-Jastrow electron-move path.

This module produces DATA ONLY (geometries, basis tables, MO coefficients, Jastrow
parameters, initial walker positions).  It holds none of the method's arithmetic: no
basis-function evaluation, no determinants, no Jastrow sums, no RNG of the move loop.
It is the one module shared by the CPU oracle (``oracle/``) and the CUDA path
(``paper_2504_07948_b200/``); those two never import each other.

Recipe: BASELINE.json ``configs[0..4]`` with the readings of SURVEY.md section 8(c).3
(A1 five-component d shells, A2 electron count, A3 normalisation, A4 Euclidean QR,
A14 electron placement, A15 lattice, A16 tree growth, A17 units, A20 per-walker
sub-streams).  The paper's own workloads (SPICE2/ccECP molecules, PAPER.md L80-86,
L259-285) are not available; these synthetic systems stand in for them and keep the
shapes (3 contracted functions per electron, 3-primitive s/p/d shells, closed-shell
single determinant, Pade Jastrow, tau 0.002-0.01).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

MASTER_SEED = 7948
ANGSTROM = 1.0 / 0.529177210903  # bohr per angstrom (A17)

# purposes for SeedSequence([seed, config, purpose, ...])
_P_GEOM, _P_BASIS, _P_MO, _P_INIT, _P_SPECIES = 1, 2, 3, 4, 5

# shells per atom kind: heavy atoms 3s2p1d, hydrogen 2s1p (BASELINE.json configs[0], [3])
_SHELLS_HEAVY = (0, 0, 0, 1, 1, 2)
_SHELLS_H = (0, 0, 1)
N_PRIM = 3


@dataclass
class System:
    """Immutable description of a molecule + trial wave function (all bohr / hartree)."""

    name: str
    atoms_xyz: np.ndarray  # [N_a, 3] float64
    Z: np.ndarray  # [N_a] float64 (charge used by e-n Jastrow and Coulomb V)
    shell_atom: np.ndarray  # [N_sh] int32
    shell_l: np.ndarray  # [N_sh] int32 in {0,1,2}
    shell_nprim: np.ndarray  # [N_sh] int32
    shell_prim_offset: np.ndarray  # [N_sh] int32
    alpha: np.ndarray  # [sum nprim] float64
    coef: np.ndarray  # [sum nprim] float64, includes ALL normalisation
    n_basis: int
    n_up: int
    n_dn: int
    C_up: np.ndarray  # [N_b, n_up] row-major float64
    C_dn: np.ndarray  # [N_b, n_dn]
    a_anti: float = 0.5
    a_para: float = 0.25
    b_ee: float = 1.0
    b_en: float = 1.0
    electron_atom: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))  # [N_e] centre of each electron's initial Gaussian

    @property
    def n_atoms(self) -> int:
        return int(self.atoms_xyz.shape[0])

    @property
    def n_shells(self) -> int:
        return int(self.shell_l.shape[0])

    @property
    def n_elec(self) -> int:
        return self.n_up + self.n_dn


@dataclass
class Workload:
    """A system plus the run parameters of one BASELINE.json config."""

    config: int
    system: System
    n_walkers: int
    tau: float
    n_sweeps: int
    delay_k: int
    seed: int = MASTER_SEED

    def positions(self, w0: int = 0, w1: int | None = None) -> np.ndarray:
        """Initial positions [w1-w0, N_e, 3] of global walkers w0..w1-1 (A14, A20)."""
        if w1 is None:
            w1 = self.n_walkers
        return initial_positions(self.system, self.config, range(w0, w1), self.seed)

    @property
    def n_moves(self) -> int:
        return self.n_walkers * self.system.n_elec * self.n_sweeps


# --------------------------------------------------------------------------- basis

def _prim_norm(alpha: float, l: int) -> float:
    # normalised primitive w.r.t. Racah-normalised solid harmonics
    return math.sqrt((2 * l + 1) / (4 * math.pi) * 2.0 * (2.0 * alpha) ** (l + 1.5) / math.gamma(l + 1.5))


def contract_normalised(alpha, raw_c, l):
    """d_p = c_p N_p / sqrt(s) so that every function of the shell has unit self-overlap (A3)."""
    alpha = np.asarray(alpha, np.float64)
    raw_c = np.asarray(raw_c, np.float64)
    Np = np.array([_prim_norm(a, l) for a in alpha])
    cn = raw_c * Np
    s = 0.0
    for p in range(len(alpha)):
        for q in range(len(alpha)):
            s += cn[p] * cn[q] * (4 * math.pi / (2 * l + 1)) * math.gamma(l + 1.5) / (
                2.0 * (alpha[p] + alpha[q]) ** (l + 1.5))
    return cn / math.sqrt(s)


def n_functions(l: int) -> int:
    return 2 * l + 1  # A1: 5-component d shells


def _make_basis(is_h: np.ndarray, rng: np.random.Generator):
    shell_atom, shell_l, alpha, coef = [], [], [], []
    for a, h in enumerate(is_h):
        for l in (_SHELLS_H if h else _SHELLS_HEAVY):
            al = 10.0 ** rng.uniform(-1.0, 2.0, N_PRIM)
            c = rng.uniform(0.1, 1.0, N_PRIM)
            shell_atom.append(a)
            shell_l.append(l)
            alpha.append(al)
            coef.append(contract_normalised(al, c, l))
    shell_l = np.asarray(shell_l, np.int32)
    n_sh = len(shell_l)
    nprim = np.full(n_sh, N_PRIM, np.int32)
    off = (np.arange(n_sh, dtype=np.int32) * N_PRIM).astype(np.int32)
    n_basis = int(sum(n_functions(int(l)) for l in shell_l))
    return (np.asarray(shell_atom, np.int32), shell_l, nprim, off,
            np.concatenate(alpha), np.concatenate(coef), n_basis)


def _orthonormal_mos(n_basis: int, n_s: int, rng: np.random.Generator) -> np.ndarray:
    """Euclidean QR of a seeded N(0,1) matrix, sign-fixed so diag(R) > 0 (A4)."""
    if n_s == 0:
        return np.zeros((n_basis, 0))
    G = rng.standard_normal((n_basis, n_s))
    Q, R = np.linalg.qr(G)
    Q = Q * np.sign(np.diag(R))[None, :]
    return np.ascontiguousarray(Q)


# --------------------------------------------------------------------------- geometry

_WATER = np.array([[0.0, 0.0, 0.0], [1.43, 1.11, 0.0], [-1.43, 1.11, 0.0]])  # bohr, configs[0]


def _random_rotation(rng: np.random.Generator) -> np.ndarray:
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def _water_cluster(n_water: int, rng: np.random.Generator):
    n = 1
    while n ** 3 < n_water:
        n += 1
    xyz, Z, is_h = [], [], []
    count = 0
    for ix in range(n):
        for iy in range(n):
            for iz in range(n):
                if count >= n_water:
                    break
                site = np.array([ix, iy, iz], float) * 3.1 * ANGSTROM
                o = site + rng.uniform(-0.3, 0.3, 3) * ANGSTROM
                Rm = _random_rotation(rng)
                mol = _WATER @ Rm.T + o
                xyz.append(mol)
                Z += [6.0, 1.0, 1.0]
                is_h += [False, True, True]
                count += 1
    return np.concatenate(xyz), np.asarray(Z), np.asarray(is_h)


def _fragment(n_atoms: int, cfg: int, seed: int):
    rng = np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_GEOM]))
    srng = np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_SPECIES]))
    counts = {"C": 300, "N": 80, "O": 100, "H": 520}
    scale = n_atoms / 1000.0
    species = []
    for s, c in counts.items():
        species += [s] * int(round(c * scale))
    species = species[:n_atoms] + ["H"] * max(0, n_atoms - len(species))
    species = list(srng.permutation(species))
    zeff = {"C": 4.0, "N": 5.0, "O": 6.0, "H": 1.0}
    xyz = np.zeros((n_atoms, 3))
    for a in range(1, n_atoms):
        while True:
            parent = int(rng.integers(0, a))
            d = rng.uniform(1.1, 1.5) * ANGSTROM
            v = rng.standard_normal(3)
            v /= np.linalg.norm(v)
            cand = xyz[parent] + d * v
            if np.min(np.linalg.norm(xyz[:a] - cand, axis=1)) >= 1.0 * ANGSTROM:
                xyz[a] = cand
                break
    Z = np.array([zeff[s] for s in species])
    is_h = np.array([s == "H" for s in species])
    return xyz, Z, is_h


def _apportion(weights: np.ndarray, total: int) -> np.ndarray:
    """Largest-remainder apportionment of `total` electrons over atoms (A2)."""
    w = np.asarray(weights, float)
    quota = w * total / w.sum()
    base = np.floor(quota).astype(int)
    rem = total - int(base.sum())
    order = np.argsort(-(quota - base), kind="stable")
    base[order[:rem]] += 1
    return base


def _electron_atoms(n_per_atom: np.ndarray, n_up: int, n_dn: int) -> np.ndarray:
    """A14: list L = atom a repeated n_a times; up p at L[2p], down p at L[2p+1]."""
    L = np.repeat(np.arange(len(n_per_atom)), n_per_atom)
    assert len(L) == n_up + n_dn
    if n_dn == 0:
        return L.astype(np.int32)
    assert n_up == n_dn
    return np.concatenate([L[0::2], L[1::2]]).astype(np.int32)


def initial_positions(system: System, cfg: int, walkers, seed: int = MASTER_SEED) -> np.ndarray:
    out = np.empty((len(walkers), system.n_elec, 3))
    centres = system.atoms_xyz[system.electron_atom]
    for n, w in enumerate(walkers):
        rng = np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_INIT, int(w)]))
        out[n] = centres + rng.standard_normal((system.n_elec, 3))
    return out


# --------------------------------------------------------------------------- systems

def _assemble(name, cfg, seed, xyz, Z, is_h, n_elec_per_atom, n_up, n_dn) -> System:
    brng = np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_BASIS]))
    sa, sl, npr, off, al, cf, nb = _make_basis(is_h, brng)
    C_up = _orthonormal_mos(nb, n_up, np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_MO, 0])))
    C_dn = _orthonormal_mos(nb, n_dn, np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_MO, 1])))
    return System(name=name, atoms_xyz=np.ascontiguousarray(xyz, np.float64), Z=np.ascontiguousarray(Z, np.float64),
                  shell_atom=sa, shell_l=sl, shell_nprim=npr, shell_prim_offset=off, alpha=al, coef=cf,
                  n_basis=nb, n_up=n_up, n_dn=n_dn, C_up=C_up, C_dn=C_dn,
                  electron_atom=_electron_atoms(np.asarray(n_elec_per_atom, int), n_up, n_dn))


def water_monomer(seed: int = MASTER_SEED, cfg: int = 0) -> System:
    Z = np.array([8.0, 1.0, 1.0])
    return _assemble("water", cfg, seed, _WATER.copy(), Z, np.array([False, True, True]), [8, 1, 1], 5, 5)


def water_cluster(n_water: int, seed: int = MASTER_SEED, cfg: int = 1) -> System:
    rng = np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_GEOM]))
    xyz, Z, is_h = _water_cluster(n_water, rng)
    n_e = 8 * n_water
    return _assemble(f"water{n_water}", cfg, seed, xyz, Z, is_h, Z.astype(int), n_e // 2, n_e // 2)


def fragment(n_atoms: int = 1000, n_elec: int = 4096, seed: int = MASTER_SEED, cfg: int = 3) -> System:
    xyz, Z, is_h = _fragment(n_atoms, cfg, seed)
    per_atom = _apportion(Z, n_elec)
    return _assemble(f"fragment{n_atoms}", cfg, seed, xyz, Z, is_h, per_atom, n_elec // 2, n_elec // 2)


_CONFIG_PARAMS = {
    0: dict(n_walkers=64, tau=0.01, n_sweeps=100, delay_k=1),
    1: dict(n_walkers=512, tau=0.005, n_sweeps=50, delay_k=32),
    2: dict(n_walkers=256, tau=0.005, n_sweeps=10, delay_k=64),
    3: dict(n_walkers=64, tau=0.002, n_sweeps=5, delay_k=128),
}

_system_cache: dict = {}


def make_system(config: int, seed: int = MASTER_SEED) -> System:
    """System of BASELINE.json configs[config]; config 4 re-uses the system of config 2."""
    cfg = 2 if config == 4 else config
    key = (cfg, seed)
    if key not in _system_cache:
        if cfg == 0:
            s = water_monomer(seed, 0)
        elif cfg == 1:
            s = water_cluster(32, seed, 1)
        elif cfg == 2:
            s = water_cluster(256, seed, 2)
        elif cfg == 3:
            s = fragment(1000, 4096, seed, 3)
        else:
            raise ValueError(f"unknown config {config}")
        _system_cache[key] = s
    return _system_cache[key]


def make_workload(config: int, n_walkers: int | None = None, delay_k: int | None = None,
                  n_sweeps: int | None = None, seed: int = MASTER_SEED) -> Workload:
    """Workload of configs[config].  Config 4 = the system (and walker streams) of config 2 with
    caller-chosen n_walkers / delay_k and 5 sweeps."""
    if config == 4:
        p = dict(_CONFIG_PARAMS[2])
        p["n_sweeps"] = 5
        base_cfg = 2
    else:
        p = dict(_CONFIG_PARAMS[config])
        base_cfg = config
    if n_walkers is not None:
        p["n_walkers"] = n_walkers
    if delay_k is not None:
        p["delay_k"] = delay_k
    if n_sweeps is not None:
        p["n_sweeps"] = n_sweeps
    return Workload(config=base_cfg, system=make_system(config, seed), seed=seed, **p)


# ------------------------------------------------------- tiny systems for tests / smoke

def hydrogen_atom() -> System:
    """One up electron, one s shell with alpha=0, coef=1, C=[[1]], Z=1, b_en=0 (A23, A24):
    Psi = exp(-r), E_L = -1/2 everywhere."""
    return System(name="hydrogen", atoms_xyz=np.zeros((1, 3)), Z=np.array([1.0]),
                  shell_atom=np.array([0], np.int32), shell_l=np.array([0], np.int32),
                  shell_nprim=np.array([1], np.int32), shell_prim_offset=np.array([0], np.int32),
                  alpha=np.array([0.0]), coef=np.array([1.0]), n_basis=1, n_up=1, n_dn=0,
                  C_up=np.ones((1, 1)), C_dn=np.zeros((1, 0)), a_anti=0.5, a_para=0.25, b_ee=1.0, b_en=0.0,
                  electron_atom=np.array([0], np.int32))


def random_molecule(n_heavy: int, n_h: int, n_up: int, n_dn: int, seed: int, spread: float = 2.5,
                    cfg: int = 99) -> System:
    """Small seeded random molecule for tests: atoms N(0, spread^2), heavy Z=6, H Z=1."""
    rng = np.random.default_rng(np.random.SeedSequence([seed, cfg, _P_GEOM]))
    n_a = n_heavy + n_h
    xyz = rng.standard_normal((n_a, 3)) * spread
    is_h = np.array([False] * n_heavy + [True] * n_h)
    Z = np.where(is_h, 1.0, 6.0)
    per_atom = _apportion(Z, n_up + n_dn)
    if n_up == n_dn or n_dn == 0:
        e_atoms = per_atom
    else:
        raise ValueError("random_molecule supports closed-shell or single-spin systems")
    return _assemble(f"rand{n_heavy}h{n_h}", cfg, seed, xyz, Z, is_h, e_atoms, n_up, n_dn)


# ------------------------------------------------------------------ row f3: semi-local pseudopotential channels (data only)

@dataclass
class Ecp:
    """Non-local channels of a semi-local pseudopotential: channel c sits on atom ch_atom[c], projects on angular
    momentum ch_l[c] (0..2) and has the radial function ch_beta[c] * exp(-ch_alpha[c] r^2); atom I acts on electrons
    closer than rcut[I] (0: the atom has no non-local part)."""

    ch_atom: np.ndarray  # [n_ch] int32
    ch_l: np.ndarray  # [n_ch] int32
    ch_beta: np.ndarray  # [n_ch] float64 (hartree)
    ch_alpha: np.ndarray  # [n_ch] float64 (bohr^-2)
    rcut: np.ndarray  # [N_a] float64 (bohr)

    @property
    def n_channels(self) -> int:
        return int(self.ch_l.shape[0])


def make_ecp(system: System) -> Ecp:
    """Synthetic stand-in for the paper's ccECPs (their tables are not reproduced): heavy atoms get an
    s channel 12 exp(-8 r^2) and a p channel -4 exp(-6 r^2), cut at 1.4 bohr; hydrogens an s channel 2 exp(-10 r^2), cut
    at 1.0 bohr.  The magnitudes, the one-Gaussian-per-channel shape and the 1-1.5 bohr range are those of first-row
    ccECP-like potentials; about one to two electrons per heavy atom sit inside the cut-off."""
    ch_atom, ch_l, beta, alpha = [], [], [], []
    rcut = np.zeros(system.n_atoms)
    for a in range(system.n_atoms):
        if system.Z[a] > 1.5:
            ch_atom += [a, a]; ch_l += [0, 1]; beta += [12.0, -4.0]; alpha += [8.0, 6.0]
            rcut[a] = 1.4
        else:
            ch_atom += [a]; ch_l += [0]; beta += [2.0]; alpha += [10.0]
            rcut[a] = 1.0
    return Ecp(np.array(ch_atom, np.int32), np.array(ch_l, np.int32), np.array(beta), np.array(alpha), rcut)


def one_orbital_atom(l: int, m: int, zeta: float = 0.7, b_en: float = 0.5) -> System:
    """One up electron on one atom at the origin in the single orbital S_lm(r) exp(-zeta r^2) (one shell of angular
    momentum l, C picks component m) with an electron-nucleus Jastrow: under a rotation about the nucleus the wave
    function transforms like S_lm alone, which makes the non-local energy a closed form (tests of row f3)."""
    nf = 2 * l + 1
    C = np.zeros((nf, 1))
    C[m, 0] = 1.0
    return System(name=f"atom_l{l}m{m}", atoms_xyz=np.zeros((1, 3)), Z=np.array([1.0]),
                  shell_atom=np.array([0], np.int32), shell_l=np.array([l], np.int32),
                  shell_nprim=np.array([1], np.int32), shell_prim_offset=np.array([0], np.int32),
                  alpha=np.array([zeta]), coef=np.array([1.0]), n_basis=nf, n_up=1, n_dn=0,
                  C_up=C, C_dn=np.zeros((nf, 0)), a_anti=0.5, a_para=0.25, b_ee=1.0, b_en=b_en,
                  electron_atom=np.array([0], np.int32))
