"""Seeded synthetic inputs for the five BASELINE.json configs.

This module only *draws inputs* (geometry, basis-set parameters, matrices).  It holds
none of the method's arithmetic (no Coulomb integrals, no Boys function, no
derivatives); both the CUDA path and the oracle receive the arrays generated here.
The recipe is stated in DESIGN.md ("Input recipe") and follows SURVEY.md §8(d):

    draw order  geometry -> heavy-atom Z -> per-shell exponents -> per-shell weights
                -> R_A -> D -> c_aux -> d_aux -> C_occ -> C_vir -> B

All lengths leave this module in bohr; all arrays are float64 / int32, C-contiguous.
The paper's own molecules (GPU4PySCF benchmark set, Table 1) and basis
data (def2-TZVP; ris exponents of Ref. 87) are not
available; these inputs take their sizes and shell structure and stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

ANGSTROM = 1.0 / 0.529177210903  # bohr per Angstrom

HEAVY_SPD = (0, 0, 0, 1, 1, 2)            # 3s2p1d
HYDROGEN = (0, 0, 1)                      # 2s1p
HEAVY_SPDF = (0, 0, 0, 0, 1, 1, 1, 2, 2, 3)  # 4s3p2d1f
NPRIM = 3


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


@dataclass
class Molecule:
    """Geometry + contracted Cartesian shells + one s-type auxiliary Gaussian per atom."""
    coords: np.ndarray          # [natoms][3] bohr
    Z: np.ndarray               # [natoms] int32 (only used to count electrons)
    shell_atom: np.ndarray      # [nshells] int32
    shell_l: np.ndarray         # [nshells] int32, 0..3
    shell_nprim: np.ndarray     # [nshells] int32
    shell_prim_off: np.ndarray  # [nshells] int32, offset into prim_exp / prim_coef
    prim_exp: np.ndarray        # [nprim_total] bohr^-2
    prim_coef: np.ndarray       # [nprim_total], applied as-is to unnormalised primitives
    aux_exponents: np.ndarray   # [natoms] bohr^-2; aux P sits on atom P
    # optional J-fit auxiliary set with p functions (NEXT-2): SHELLS (atom[], l[] in {0, 1}, exponent[]);
    # None: the J term uses the default set above
    jfit: tuple | None = None

    @property
    def natoms(self) -> int:
        return int(self.coords.shape[0])

    @property
    def nshells(self) -> int:
        return int(self.shell_l.shape[0])

    @property
    def nao(self) -> int:
        return int(sum(ncart(int(l)) for l in self.shell_l))

    @property
    def ao_off(self) -> np.ndarray:
        n = np.array([ncart(int(l)) for l in self.shell_l], dtype=np.int64)
        return np.concatenate([[0], np.cumsum(n)[:-1]]).astype(np.int32)

    @property
    def ao_atom(self) -> np.ndarray:
        out = []
        for s in range(self.nshells):
            out += [int(self.shell_atom[s])] * ncart(int(self.shell_l[s]))
        return np.array(out, dtype=np.int32)


@dataclass
class Workload:
    name: str
    mol: Molecule
    nocc: int
    nvir: int
    D: np.ndarray        # [nbatch_J][nao][nao]
    c_aux: np.ndarray    # [nbatch_J][naux]
    d_aux: np.ndarray    # [nbatch_J][naux]
    C_occ: np.ndarray    # [nao][nocc]
    C_vir: np.ndarray    # [nao][nvir]
    B: np.ndarray        # [nbatch_K][naux][nocc][nvir]
    schwarz_tol: float = 1e-13
    meta: dict = field(default_factory=dict)


# ----------------------------------------------------------------------------- geometry

def _triatomic() -> tuple[np.ndarray, list[bool]]:
    r = 0.96
    th = math.radians(104.5)
    xyz = np.array([[0.0, 0.0, 0.0],
                    [r, 0.0, 0.0],
                    [r * math.cos(th), r * math.sin(th), 0.0]])
    return xyz, [True, False, False]


def _blob(rng: np.random.Generator, nheavy: int, nh: int) -> tuple[np.ndarray, list[bool]]:
    """Heavy atoms on a jittered 1.4 A cubic grid (connected blob), H caps at 1.09 A."""
    step = 1.4
    sites = [(0, 0, 0)]
    occupied = {(0, 0, 0)}
    dirs = [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    while len(sites) < nheavy:
        base = sites[int(rng.integers(len(sites)))]
        d = dirs[int(rng.integers(6))]
        new = (base[0] + d[0], base[1] + d[1], base[2] + d[2])
        if new not in occupied:
            occupied.add(new)
            sites.append(new)
    heavy = np.array(sites, dtype=np.float64) * step
    heavy += rng.uniform(-0.15, 0.15, size=heavy.shape)
    # jitter keeps neighbours >= 1.1 A apart; checked anyway
    for i in range(nheavy):
        dd = np.linalg.norm(heavy[i + 1:] - heavy[i], axis=1)
        assert dd.size == 0 or dd.min() >= 1.0
    atoms = [h for h in heavy]
    hosts = rng.permutation(nheavy)[:nh]
    for host in hosts:
        for _ in range(10000):
            v = rng.normal(size=3)
            v /= np.linalg.norm(v)
            cand = heavy[host] + 1.09 * v
            dist = np.linalg.norm(np.array(atoms) - cand, axis=1)
            dist_ok = np.sum(dist < 1.0) == 0
            if dist_ok:
                atoms.append(cand)
                break
        else:
            raise RuntimeError("could not place a hydrogen")
    return np.array(atoms), [True] * nheavy + [False] * nh


def _chain(nback: int) -> tuple[np.ndarray, list[bool]]:
    """Planar zig-zag backbone (bond 1.4 A, angle 120 deg), one in-plane H per atom."""
    dx = 1.4 * math.sin(math.radians(60.0))
    dy = 1.4 * math.cos(math.radians(60.0))
    back = np.zeros((nback, 3))
    hyd = np.zeros((nback, 3))
    for i in range(nback):
        s = 1.0 if i % 2 == 0 else -1.0
        back[i] = (i * dx, s * dy / 2.0, 0.0)
        hyd[i] = (i * dx, s * (dy / 2.0 + 1.09), 0.0)
    return np.concatenate([back, hyd]), [True] * nback + [False] * nback


# ----------------------------------------------------------------------------- basis

def _dfact2(l: int) -> float:
    """(2l-1)!!"""
    out = 1.0
    for k in range(1, 2 * l, 2):
        out *= k
    return out


def _make_shell(rng: np.random.Generator, l: int, lo: float, hi: float):
    a = np.exp(rng.uniform(math.log(lo), math.log(hi), size=NPRIM))
    return l, a


def _contract(l: int, a: np.ndarray, w: np.ndarray) -> np.ndarray:
    """d_k = w_k (2a/pi)^{3/4} (4a)^{l/2} / sqrt((2l-1)!!), then scale the shell so that the
    x^l component has unit self-overlap."""
    d = w * (2.0 * a / math.pi) ** 0.75 * (4.0 * a) ** (l / 2.0) / math.sqrt(_dfact2(l))
    s = 0.0
    for j in range(len(a)):
        for k in range(len(a)):
            g = a[j] + a[k]
            s += d[j] * d[k] * _dfact2(l) / (2.0 * g) ** l * (math.pi / g) ** 1.5
    return d / math.sqrt(s)


def _build_molecule(rng, xyz_ang, is_heavy, heavy_shells, lo, hi) -> Molecule:
    natoms = len(is_heavy)
    Z = np.array([int(rng.integers(6, 9)) if h else 1 for h in is_heavy], dtype=np.int32)
    shells = []
    for A in range(natoms):
        for l in (heavy_shells if is_heavy[A] else HYDROGEN):
            shells.append((A,) + _make_shell(rng, l, lo, hi))
    weights = [rng.uniform(0.2, 1.0, size=NPRIM) for _ in shells]
    shell_atom = np.array([s[0] for s in shells], dtype=np.int32)
    shell_l = np.array([s[1] for s in shells], dtype=np.int32)
    shell_nprim = np.full(len(shells), NPRIM, dtype=np.int32)
    shell_prim_off = (np.arange(len(shells)) * NPRIM).astype(np.int32)
    prim_exp = np.concatenate([s[2] for s in shells])
    prim_coef = np.concatenate([_contract(s[1], s[2], w) for s, w in zip(shells, weights)])
    R_A = rng.uniform(0.6, 1.8, size=natoms) * ANGSTROM
    aux = 0.2 / R_A ** 2
    return Molecule(np.ascontiguousarray(xyz_ang * ANGSTROM), Z, shell_atom, shell_l, shell_nprim,
                    shell_prim_off, prim_exp, prim_coef, aux)


# ----------------------------------------------------------------------------- configs

CONFIG_NAMES = {
    1: "config1-triatomic-25ao",
    2: "config2-blob30-300ao",
    3: "config3-blob100-1100ao",
    4: "config4-chain300-3000ao",
    5: "config5-spdf40-1400ao",
}


def make_molecule(config: int) -> tuple[Molecule, np.random.Generator]:
    seed = config - 1
    rng = np.random.default_rng(seed)
    if config == 1:
        xyz, heavy = _triatomic()
        mol = _build_molecule(rng, xyz, heavy, HEAVY_SPD, 0.1, 50.0)
        # config 1 draws no Z for nocc: nocc is fixed at 5
    elif config == 2:
        xyz, heavy = _blob(rng, 15, 15)
        mol = _build_molecule(rng, xyz, heavy, HEAVY_SPD, 0.1, 50.0)
    elif config == 3:
        xyz, heavy = _blob(rng, 60, 40)
        mol = _build_molecule(rng, xyz, heavy, HEAVY_SPD, 0.1, 50.0)
    elif config == 4:
        xyz, heavy = _chain(150)
        mol = _build_molecule(rng, xyz, heavy, HEAVY_SPD, 0.1, 50.0)
        mol.Z[:150] = 6   # backbone is carbon-like
    elif config == 5:
        xyz, heavy = _blob(rng, 40, 0)
        mol = _build_molecule(rng, xyz, heavy, HEAVY_SPDF, 0.05, 200.0)
    else:
        raise ValueError("config must be 1..5")
    return mol, rng


def make_workload(config: int, *, nbatch_override: int | None = None,
                  with_B: bool = True) -> Workload:
    """Full seeded workload of BASELINE.json config `config` (1-based).

    nbatch: config 1 -> 1; config 2 -> J 2 (one symmetric D, one
    non-symmetric), K 1; config 3 -> 5; config 4 -> 3 (two states + one non-symmetric
    derivative-coupling contraction); config 5 -> 1.
    """
    mol, rng = make_molecule(config)
    nao, naux = mol.nao, mol.natoms
    if config == 1:
        nocc, nvir = 5, 20
    else:
        nocc = int(mol.Z.sum()) // 2
        nvir = min(nao - nocc, 2 * nocc)
    nbJ = {1: 1, 2: 2, 3: 5, 4: 3, 5: 1}[config]
    nbK = {1: 1, 2: 1, 3: 5, 4: 3, 5: 1}[config]
    if nbatch_override is not None:
        nbJ = nbK = nbatch_override
    D = rng.standard_normal((nbJ, nao, nao))
    if config == 2:
        D[0] = 0.5 * (D[0] + D[0].T)          # symmetric; D[1] stays non-symmetric ("X+Y")
    elif config in (3, 5):
        D = 0.5 * (D + D.transpose(0, 2, 1))
    elif config == 4:
        D[:2] = 0.5 * (D[:2] + D[:2].transpose(0, 2, 1))   # D[2]: transition density
    c_aux = rng.standard_normal((nbJ, naux))
    d_aux = rng.standard_normal((nbJ, naux))
    C_occ = rng.standard_normal((nao, nocc))
    C_vir = rng.standard_normal((nao, nvir))
    if with_B:
        B = rng.standard_normal((nbK, naux, nocc, nvir))
    else:
        B = np.zeros((0, naux, nocc, nvir))
    return Workload(CONFIG_NAMES[config], mol, nocc, nvir, np.ascontiguousarray(D), c_aux, d_aux,
                    C_occ, C_vir, B, 1e-13,
                    {"config": config, "seed": config - 1, "nao": nao, "naux": naux,
                     "nbatch_J": nbJ, "nbatch_K": nbK})


def with_jfit(mol: Molecule, seed: int, p_on=None) -> Molecule:
    """A copy of `mol` carrying a J-fit set of one s shell (the default exponent) and one p shell per atom -- the set the
    paper's calculations use for the Coulomb term.  The paper's fitted exponents (Ref. 87) are
    not available: the p exponent is the atom's s exponent times a seeded factor in [0.8, 2.0].  p_on: atoms that get the
    p shell (default all)."""
    import copy
    rng = np.random.default_rng(seed)
    fac = rng.uniform(0.8, 2.0, size=mol.natoms)
    at, ll, ex = [], [], []
    for A in range(mol.natoms):
        at.append(A); ll.append(0); ex.append(float(mol.aux_exponents[A]))
        if p_on is None or A in p_on:
            at.append(A); ll.append(1); ex.append(float(mol.aux_exponents[A] * fac[A]))
    out = copy.copy(mol)
    out.jfit = (np.array(at, dtype=np.int32), np.array(ll, dtype=np.int32), np.array(ex, dtype=np.float64))
    return out


def naux_jfit(mol: Molecule) -> int:
    if mol.jfit is None:
        return mol.natoms
    return int(sum(3 if l else 1 for l in mol.jfit[1]))


def tiny_molecule(seed: int, ls_per_atom, coords_bohr, lo=0.2, hi=3.0, nprim=2) -> Molecule:
    """Small hand-shaped molecule for unit tests: `ls_per_atom[A]` lists shell l values."""
    rng = np.random.default_rng(seed)
    coords = np.ascontiguousarray(np.asarray(coords_bohr, dtype=np.float64))
    natoms = coords.shape[0]
    sa, sl, sn, so, ex, co = [], [], [], [], [], []
    off = 0
    for A in range(natoms):
        for l in ls_per_atom[A]:
            a = np.exp(rng.uniform(math.log(lo), math.log(hi), size=nprim))
            w = rng.uniform(0.2, 1.0, size=nprim)
            sa.append(A); sl.append(l); sn.append(nprim); so.append(off)
            ex.append(a); co.append(_contract(l, a, w))
            off += nprim
    aux = rng.uniform(0.05, 0.6, size=natoms)
    return Molecule(coords, np.ones(natoms, dtype=np.int32),
                    np.array(sa, dtype=np.int32), np.array(sl, dtype=np.int32),
                    np.array(sn, dtype=np.int32), np.array(so, dtype=np.int32),
                    np.concatenate(ex), np.concatenate(co), aux)
