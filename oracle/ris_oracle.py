"""ctypes front end of the CPU oracle (oracle/ris_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It imports nothing from paper_2511_18233_b200 except that callers hand
it a `synth.Molecule`-shaped object (duck-typed: coords, shell_*, prim_*, aux_exponents).

What it computes (Eq. 27 terms 1-3 with everything that is not an integral
derivative folded into the inputs; Eqs. 21-22 for the integrals):

    grad_J (mol, D, c)              -> G_J[s,A,x] = sum_{mu nu P} D^s_{mu nu} c^s_P d(mu nu|P)/dR_A
    grad_K (mol, C_occ, C_vir, B)   -> G_K[s,A,x] = sum_P sum_{mu nu} Gamma^{s,P}_{mu nu} d(mu nu|P)/dR_A
                                       Gamma^{s,P} = C_occ B[s,P] C_vir^T   (numpy float64 matmul,
                                       i.e. the host BLAS that numpy links; stated in DESIGN.md)
    grad_PQ(mol, c, d)              -> G_PQ[s,A,x] = sum_{PQ} c_P d_Q d(P|Q)/dR_A

Each also returns the undifferentiated scalar (E_J, E_K, E_PQ) used by the finite-difference pin.
`atoms=` samples the output: only rows of the listed atoms are computed (and returned; the other
rows are NaN), visiting only triplets that touch them -- the definition restricted to those
outputs, used for full-size parity.  `aux=` restricts the sum over P to the listed auxiliary
functions (a bounded sample of the same workload, used only for timing the oracle in bench.py).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libris_oracle.so")
_SRC = os.path.join(_HERE, "ris_oracle.c")
_lib = None


_SO_EXT = os.path.join(_HERE, "libris_oracle_ext.so")


def build(force: bool = False, extended: bool = False) -> str:
    """gcc -O2 -fopenmp -shared.  No -ffast-math: IEEE semantics, long double accumulators.
    extended=True builds the SAME source with every intermediate in `long double` (-DORACLE_REAL): not the oracle,
    but the yardstick tests/test_oracle_pins.py measures the oracle's own FP64 rounding error with."""
    so = _SO_EXT if extended else _SO
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=gnu99", "-fopenmp", "-fPIC", "-shared"]
                              + (['-DORACLE_REAL=long double'] if extended else []) + ["-o", so, _SRC, "-lm"])
    return so


class _Mol(C.Structure):
    _fields_ = [("natoms", C.c_int), ("coords", C.c_void_p), ("nshells", C.c_int),
                ("shell_atom", C.c_void_p), ("shell_l", C.c_void_p), ("shell_nprim", C.c_void_p),
                ("shell_prim_off", C.c_void_p), ("prim_exp", C.c_void_p), ("prim_coef", C.c_void_p),
                ("aux_exponents", C.c_void_p),
                # explicit auxiliary function list (NEXT-2: the J-fit set with p functions); naux_fn = 0: default set
                ("naux_fn", C.c_int), ("aux_atom", C.c_void_p), ("aux_l", C.c_void_p), ("aux_comp", C.c_void_p),
                ("aux_exp", C.c_void_p)]


class extended_precision:
    """`with extended_precision(): ...` routes every call of this module to the long-double-intermediate build."""

    def __enter__(self):
        global _lib
        self._saved = _lib
        _lib = None
        _load(build(extended=True))

    def __exit__(self, *exc):
        global _lib
        _lib = self._saved


def lib():
    if _lib is None:
        _load(build())
    return _lib


def _load(so):
    global _lib
    if True:
        _lib = C.CDLL(so)
        _lib.ris_oracle_boys.argtypes = [C.c_int, C.c_double, C.c_void_p]
        _lib.ris_oracle_prim3c.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double,
                                           C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.ris_oracle_prim2c.argtypes = [C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.ris_oracle_prim3c_aux.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double,
                                               C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        _lib.ris_oracle_prim2c_lm.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                              C.c_void_p, C.c_void_p]
        _lib.ris_oracle_contract_P.argtypes = [C.POINTER(_Mol), C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                               C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        _lib.ris_oracle_contract_P.restype = C.c_int
        _lib.ris_oracle_grad_PQ.argtypes = [C.POINTER(_Mol), C.c_int, C.c_void_p, C.c_void_p,
                                            C.c_void_p, C.c_void_p]
        _lib.ris_oracle_int3c_P.argtypes = [C.POINTER(_Mol), C.c_int, C.c_double, C.c_void_p]
        _lib.ris_oracle_int3c_P.restype = C.c_int
        _lib.ris_oracle_num_threads.restype = C.c_int


def num_threads() -> int:
    return int(lib().ris_oracle_num_threads())


def _f64(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _i32(x):
    return np.ascontiguousarray(x, dtype=np.int32)


def jfit_functions(mol):
    """The J-fit auxiliary FUNCTIONS of `mol` as arrays (atom, l, component, exponent), or None when the molecule carries
    no explicit J-fit set (then J and K share the default set: one s function per atom).  mol.jfit = (atom[], l[], exp[])
    lists auxiliary SHELLS with l in {0, 1}; a p shell expands into its x, y, z components, in that order."""
    jf = getattr(mol, "jfit", None)
    if jf is None:
        return None
    at, ll, ex = (np.asarray(x) for x in jf)
    fa, fl, fc, fe = [], [], [], []
    for a, l, e in zip(at, ll, ex):
        assert int(l) in (0, 1), "auxiliary shells are s or p"
        for comp in range(1 if int(l) == 0 else 3):
            fa.append(int(a)); fl.append(int(l)); fc.append(comp); fe.append(float(e))
    return _i32(fa), _i32(fl), _i32(fc), _f64(fe)


class _Held:
    """Keeps the numpy buffers alive next to the C struct.  jfit=True: the J-type calls see the molecule's J-fit auxiliary
    set (if it has one); the K-type calls always see the default set."""

    def __init__(self, mol, jfit=False):
        self.aux = jfit_functions(mol) if jfit else None
        self.arrs = dict(coords=_f64(mol.coords), shell_atom=_i32(mol.shell_atom), shell_l=_i32(mol.shell_l),
                         shell_nprim=_i32(mol.shell_nprim), shell_prim_off=_i32(mol.shell_prim_off),
                         prim_exp=_f64(mol.prim_exp), prim_coef=_f64(mol.prim_coef),
                         aux_exponents=_f64(mol.aux_exponents))
        a = self.arrs
        self.natoms = a["coords"].shape[0]
        self.nao = int(sum((l + 1) * (l + 2) // 2 for l in a["shell_l"]))
        self.ao_atom = np.concatenate([[int(at)] * ((l + 1) * (l + 2) // 2)
                                       for at, l in zip(a["shell_atom"], a["shell_l"])]).astype(np.int64)
        self.c = _Mol(self.natoms, a["coords"].ctypes.data, a["shell_l"].shape[0], a["shell_atom"].ctypes.data,
                      a["shell_l"].ctypes.data, a["shell_nprim"].ctypes.data, a["shell_prim_off"].ctypes.data,
                      a["prim_exp"].ctypes.data, a["prim_coef"].ctypes.data, a["aux_exponents"].ctypes.data,
                      0, None, None, None, None)
        self.naux = self.natoms
        if self.aux is not None:
            fa, fl, fc, fe = self.aux
            self.naux = int(fa.shape[0])
            self.c.naux_fn = self.naux
            self.c.aux_atom, self.c.aux_l, self.c.aux_comp, self.c.aux_exp = (x.ctypes.data for x in (fa, fl, fc, fe))


def boys(mmax: int, T: float) -> np.ndarray:
    out = np.zeros(mmax + 1)
    lib().ris_oracle_boys(mmax, float(T), out.ctypes.data)
    return out


def prim3c(la, lb, a, b, alpha, A, B, Cc) -> np.ndarray:
    """[value, dA(3), dB(3), dC(3)] of the unnormalised primitive integral, no N_P."""
    la, lb = _i32(la), _i32(lb)
    A, B, Cc = _f64(A), _f64(B), _f64(Cc)
    out = np.zeros(10)
    lib().ris_oracle_prim3c(la.ctypes.data, lb.ctypes.data, a, b, alpha, A.ctypes.data, B.ctypes.data,
                            Cc.ctypes.data, out.ctypes.data)
    return out


def prim3c_aux(la, lb, a, b, alpha, A, B, Cc, aux_l, aux_comp) -> np.ndarray:
    """As prim3c for an unnormalised auxiliary primitive of type aux_l (0: s; 1: p, component aux_comp)."""
    la, lb = _i32(la), _i32(lb)
    A, B, Cc = _f64(A), _f64(B), _f64(Cc)
    out = np.zeros(10)
    lib().ris_oracle_prim3c_aux(la.ctypes.data, lb.ctypes.data, a, b, alpha, A.ctypes.data, B.ctypes.data,
                                Cc.ctypes.data, int(aux_l), int(aux_comp), out.ctypes.data)
    return out


def prim2c_lm(alpha, beta, lP, iP, lQ, iQ, RP, RQ) -> np.ndarray:
    """[value, d/dR_P(3)] of the two-centre integral between unnormalised s / p auxiliary primitives."""
    RP, RQ = _f64(RP), _f64(RQ)
    out = np.zeros(4)
    lib().ris_oracle_prim2c_lm(alpha, beta, int(lP), int(iP), int(lQ), int(iQ), RP.ctypes.data, RQ.ctypes.data, out.ctypes.data)
    return out


def prim2c(alpha, beta, RP, RQ) -> np.ndarray:
    """[value, d/dR_P(3)] of (P|Q) without N_P N_Q."""
    RP, RQ = _f64(RP), _f64(RQ)
    out = np.zeros(4)
    lib().ris_oracle_prim2c(alpha, beta, RP.ctypes.data, RQ.ctypes.data, out.ctypes.data)
    return out


def _mask(natoms, atoms):
    if atoms is None:
        return None
    m = np.zeros(natoms, dtype=np.uint8)
    m[np.asarray(atoms, dtype=np.int64)] = 1
    return m


def _finish(g, e, mask):
    g = g.astype(np.float64)
    if mask is not None:
        g[:, mask == 0, :] = np.nan
        return g, None       # the scalar is not defined on a sampled run
    return g, e.astype(np.float64)


def grad_J(mol, D, c_aux, *, atoms=None, prim_cutoff=0.0, aux=None):
    """G_J and E_J = sum D_{mu nu} c_P (mu nu|P).  D [nbatch][nao][nao] (any symmetry), c [nbatch][naux]."""
    h = _Held(mol, jfit=True)
    D = _f64(D).reshape(-1, h.nao, h.nao)
    c_aux = _f64(c_aux).reshape(D.shape[0], h.naux)
    nb = D.shape[0]
    mask = _mask(h.natoms, atoms)
    g = np.zeros((nb, h.natoms, 3), dtype=np.longdouble)
    e = np.zeros(nb, dtype=np.longdouble)
    for P in (range(h.naux) if aux is None else aux):
        sc = _f64(c_aux[:, P])
        rc = lib().ris_oracle_contract_P(C.byref(h.c), P, nb, D.ctypes.data, sc.ctypes.data,
                                         mask.ctypes.data if mask is not None else None, prim_cutoff,
                                         g.ctypes.data, e.ctypes.data)
        assert rc == 0
    return _finish(g, e, mask)


def gamma_P(C_occ, C_vir, B_sP, rows=None):
    """Gamma^P = C_occ B^P C_vir^T (Eqs. 32-34, 39: AO back-transform).
    `rows`: AO indices on sampled atoms; only Gamma[rows,:] and Gamma[:,rows] are filled."""
    if rows is None:
        return C_occ @ B_sP @ C_vir.T
    nao = C_occ.shape[0]
    G = np.zeros((nao, nao))
    G[rows, :] = (C_occ[rows, :] @ B_sP) @ C_vir.T
    G[:, rows] = C_occ @ (B_sP @ C_vir[rows, :].T)
    return G


def grad_K(mol, C_occ, C_vir, B, *, atoms=None, prim_cutoff=0.0, aux=None):
    """G_K and E_K = sum_P sum Gamma^P_{mu nu} (mu nu|P).  B [nbatch][naux][nocc][nvir]."""
    h = _Held(mol)
    C_occ, C_vir = _f64(C_occ), _f64(C_vir)
    B = _f64(B).reshape(-1, h.natoms, C_occ.shape[1], C_vir.shape[1])
    nb = B.shape[0]
    mask = _mask(h.natoms, atoms)
    g = np.zeros((nb, h.natoms, 3), dtype=np.longdouble)
    e = np.zeros(nb, dtype=np.longdouble)
    one = np.ones(nb)
    rows_sampled = None if mask is None else np.nonzero(mask[h.ao_atom])[0]
    for P in (range(h.natoms) if aux is None else aux):
        rows = None if (mask is None or mask[P]) else rows_sampled
        G = _f64(np.stack([gamma_P(C_occ, C_vir, B[s, P], rows) for s in range(nb)]))
        rc = lib().ris_oracle_contract_P(C.byref(h.c), P, nb, G.ctypes.data, one.ctypes.data,
                                         mask.ctypes.data if mask is not None else None, prim_cutoff,
                                         g.ctypes.data, e.ctypes.data)
        assert rc == 0
    return _finish(g, e, mask)


def grad_PQ(mol, c_aux, d_aux):
    """G_PQ and E_PQ = sum_{PQ} c_P d_Q (P|Q) (positive sign; Eq. 27's minus is the caller's)."""
    h = _Held(mol, jfit=True)
    c_aux = _f64(c_aux).reshape(-1, h.naux)
    d_aux = _f64(d_aux).reshape(-1, h.naux)
    nb = c_aux.shape[0]
    g = np.zeros((nb, h.natoms, 3), dtype=np.longdouble)
    e = np.zeros(nb, dtype=np.longdouble)
    lib().ris_oracle_grad_PQ(C.byref(h.c), nb, c_aux.ctypes.data, d_aux.ctypes.data, g.ctypes.data, e.ctypes.data)
    return g.astype(np.float64), e.astype(np.float64)


# ------------------------------------------------------------------------------------------------
# NEXT-1: the J-type fitting step either side of the derivative path, Eqs. 21-22
# with the Coulomb pairing of Eq. 21's first term:
#   v_P   = sum_{mu nu} D_{mu nu} (mu nu|P)                        (undifferentiated three-centre contraction)
#   M_PQ  = (P|Q)  with N_P N_Q                                    (Eq. 22)
#   c     = M^-1 v                                                 (numpy.linalg.solve: a library step)
#   E_RIJ = 1/2 v^T M^-1 v = 1/2 sum_{pq,sr} D_pq (pq|A) M^-1_AB (B|sr) D_sr
# and, for fixed symmetric-or-not D, Eq. 27 gives
#   dE_RIJ/dxi = sum_P c_P v_P^xi - 1/2 c^T M^xi c = G_J(D, c) - 1/2 G_PQ(c, c).
def vec_J(mol, D, *, prim_cutoff=0.0):
    """v[s][P] = sum_{mu nu} D^s_{mu nu} (mu nu|P) over all ordered (mu, nu); P runs over the J-fit set."""
    h = _Held(mol, jfit=True)
    D = _f64(D).reshape(-1, h.nao, h.nao)
    nb = D.shape[0]
    one = np.ones(nb)
    v = np.zeros((nb, h.naux))
    for P in range(h.naux):
        g = np.zeros((nb, h.natoms, 3), dtype=np.longdouble)
        e = np.zeros(nb, dtype=np.longdouble)
        rc = lib().ris_oracle_contract_P(C.byref(h.c), P, nb, D.ctypes.data, one.ctypes.data, None, prim_cutoff,
                                         g.ctypes.data, e.ctypes.data)
        assert rc == 0
        v[:, P] = e.astype(np.float64)
    return v


def metric(mol):
    """M[P][Q] = N_P N_Q (P|Q), Eq. 22."""
    al = _f64(mol.aux_exponents)
    R = _f64(mol.coords)
    n = al.shape[0]
    N = (2.0 * al / np.pi) ** 0.75
    M = np.zeros((n, n))
    for P in range(n):
        for Q in range(n):
            M[P, Q] = N[P] * N[Q] * prim2c(al[P], al[Q], R[P], R[Q])[0]
    return M


def metric_J(mol):
    """The metric of the J-fit set: M[f][g] = N_f N_g (f|g) over s and p functions (Eq. 22; the set of
    PAPER.md:125 / 168).  Without an explicit J-fit set this is metric(mol)."""
    fn = jfit_functions(mol)
    if fn is None:
        return metric(mol)
    fa, fl, fc, fe = fn
    R = _f64(mol.coords)
    n = fa.shape[0]
    N = (2.0 * fe / np.pi) ** 0.75 * np.where(fl == 1, 2.0 * np.sqrt(fe), 1.0)
    M = np.zeros((n, n))
    for P in range(n):
        for Q in range(n):
            M[P, Q] = N[P] * N[Q] * prim2c_lm(fe[P], fe[Q], fl[P], fc[P], fl[Q], fc[Q], R[fa[P]], R[fa[Q]])[0]
    return M


def fit_J(mol, D, *, prim_cutoff=0.0):
    """(v, c, E_RIJ): c = M^-1 v, E_RIJ[s] = 1/2 v[s].c[s]; M = the J-fit metric."""
    v = vec_J(mol, D, prim_cutoff=prim_cutoff)
    c = np.linalg.solve(metric_J(mol), v.T).T
    return v, c, 0.5 * np.einsum("sp,sp->s", v, c)


def grad_RIJ(mol, D, *, prim_cutoff=0.0):
    """dE_RIJ/dR at fixed D: G_J(D, c) - 1/2 G_PQ(c, c) with the fitted c (Eq. 27)."""
    _, c, _ = fit_J(mol, D, prim_cutoff=prim_cutoff)
    gJ, _ = grad_J(mol, D, c, prim_cutoff=prim_cutoff)
    gQ, _ = grad_PQ(mol, c, c)
    return gJ - 0.5 * gQ


# ------------------------------------------------------------------------------------------------
# NEXT-1, K-type fitting step: the MO-transformed three-index tensor and its fit (Eqs. 21-22, PAPER.md:119-121;
# "transformed from the AO to the MO basis and stored in the reduced-size MO basis"):
#   T^P_ia = sum_{mu nu} C_occ[mu,i] (mu nu|P) C_vir[nu,a]
#   B      = M^-1 T                                    (per (i,a) column; numpy.linalg.solve)
#   E_RIK  = 1/2 sum_{PQ} sum_ia T^P_ia M^-1_PQ T^Q_ia = 1/2 sum_P sum_ia T^P_ia B^P_ia
# and for fixed C_occ, C_vir (Eq. 27; A9: the metric term carries the FULL matrix G, not a rank-1 one)
#   dE_RIK/dxi = G_K(C_occ, C_vir, B) - 1/2 sum_{PQ} G_PQ M^xi_PQ,   G_PQ = sum_ia B^P_ia B^Q_ia.
def int3c(mol, P, *, prim_cutoff=0.0):
    """(mu nu|P) as a dense [nao][nao] matrix."""
    h = _Held(mol)
    out = np.zeros((h.nao, h.nao))
    rc = lib().ris_oracle_int3c_P(C.byref(h.c), int(P), prim_cutoff, out.ctypes.data)
    assert rc == 0
    return out


def tensor_K(mol, C_occ, C_vir, *, prim_cutoff=0.0):
    """T[P][i][a] = sum C_occ[mu,i] (mu nu|P) C_vir[nu,a]."""
    C_occ, C_vir = _f64(C_occ), _f64(C_vir)
    n = np.asarray(mol.coords).shape[0]
    return np.stack([C_occ.T @ int3c(mol, P, prim_cutoff=prim_cutoff) @ C_vir for P in range(n)])


def fit_K(mol, C_occ, C_vir, *, prim_cutoff=0.0):
    """(T, B, E_RIK): B = M^-1 T, E_RIK = 1/2 sum T.B."""
    T = tensor_K(mol, C_occ, C_vir, prim_cutoff=prim_cutoff)
    n = T.shape[0]
    B = np.linalg.solve(metric(mol), T.reshape(n, -1)).reshape(T.shape)
    return T, B, 0.5 * float(np.sum(T * B))


def grad_PQ_full(mol, G):
    """sum_{PQ} G[s][P][Q] d(P|Q)/dR with N_P N_Q (the metric term of Eq. 27 for a full matrix G; positive sign)."""
    al = _f64(mol.aux_exponents)
    R = _f64(mol.coords)
    n = al.shape[0]
    G = _f64(G).reshape(-1, n, n)
    N = (2.0 * al / np.pi) ** 0.75
    g = np.zeros((G.shape[0], n, 3), dtype=np.longdouble)
    for P in range(n):
        for Q in range(n):
            if P == Q:
                continue
            d = N[P] * N[Q] * prim2c(al[P], al[Q], R[P], R[Q])[1:]
            for s in range(G.shape[0]):
                g[s, P] += G[s, P, Q] * d
                g[s, Q] -= G[s, P, Q] * d
    return g.astype(np.float64)


def grad_RIK(mol, C_occ, C_vir, *, prim_cutoff=0.0):
    """dE_RIK/dR at fixed C_occ, C_vir: G_K(C_occ, C_vir, B) - 1/2 G_PQ_full(B B^T) with the fitted B."""
    _, B, _ = fit_K(mol, C_occ, C_vir, prim_cutoff=prim_cutoff)
    n = B.shape[0]
    gK, _ = grad_K(mol, C_occ, C_vir, B[None], prim_cutoff=prim_cutoff)
    Bf = B.reshape(n, -1)
    return gK[0] - 0.5 * grad_PQ_full(mol, (Bf @ Bf.T)[None])[0]


# ------------------------------------------------------------------------------------------------
# NEXT-1, the composed term <g^ris,(xi); {D1, D2}> of Eqs. 25-27 for two AO matrices D1, D2
# (Eq. 38-39: <g; {D1, D2}> = sum_{pqrs} g_{pq,rs} [D1]_pq [D2]_rs), with Eq. 5 / 21 read in the
# index order of Eq. 39, g_{pq,rs} = (pq|rs) - c_x (ps|rq):
#   S(R) = sum_AB M^-1_AB ( Tr[I^A D1] Tr[I^B D2] - c_x sum_{pqrs} I^A_ps I^B_rq D1_pq D2_rs ),   I^A_pq = (pq|A)
# written out in the AO basis with dense matrices (tiny molecules only).  Its derivative at FIXED D1, D2 by Eq. 27:
#   J part:  G_J(D1, c2) + G_J(D2, c1) - G_PQ(c1, c2),                c_i = M^-1 Tr[I D_i]
#   K part:  sum_A <I^A,xi; G1^A + G2^A> - sum_CD N_CD M^xi_CD,
#            G1^A = sum_B M^-1_AB D1 I^B D2,  G2^A = sum_B M^-1_AB D1^T I^B D2^T,  N = M^-1 K M^-1,
#            K_AB = sum_ps I^A_ps (D1 I^B D2)_ps.
def ris_pair_scalar(mol, D1, D2, c_x):
    n = np.asarray(mol.coords).shape[0]
    I = [int3c(mol, P) for P in range(n)]
    Minv = np.linalg.inv(metric(mol))
    v1 = np.array([np.sum(I[A] * D1) for A in range(n)])
    v2 = np.array([np.sum(I[A] * D2) for A in range(n)])
    K = np.array([[np.sum(I[A] * (D1 @ I[B] @ D2)) for B in range(n)] for A in range(n)])
    return float(v1 @ Minv @ v2 - c_x * np.sum(Minv * K))


def grad_dense_K(mol, G):
    """sum_P sum_{mu nu} G[P][mu][nu] d(mu nu|P)/dR for dense AO matrices G[P] (the K-type contraction of
    ris_oracle_contract_P with the matrices given directly)."""
    h = _Held(mol)
    G = _f64(G).reshape(h.natoms, h.nao, h.nao)
    g = np.zeros((1, h.natoms, 3), dtype=np.longdouble)
    e = np.zeros(1, dtype=np.longdouble)
    one = np.ones(1)
    for P in range(h.natoms):
        GP = _f64(G[P])
        rc = lib().ris_oracle_contract_P(C.byref(h.c), P, 1, GP.ctypes.data, one.ctypes.data, None, 0.0,
                                         g.ctypes.data, e.ctypes.data)
        assert rc == 0
    return g.astype(np.float64)[0]


def ris_pair_gradient(mol, D1, D2, c_x):
    n = np.asarray(mol.coords).shape[0]
    I = [int3c(mol, P) for P in range(n)]
    Minv = np.linalg.inv(metric(mol))
    v1 = np.array([np.sum(I[A] * D1) for A in range(n)])
    v2 = np.array([np.sum(I[A] * D2) for A in range(n)])
    c1, c2 = Minv @ v1, Minv @ v2
    gJ = grad_J(mol, D1[None], c2[None])[0][0] + grad_J(mol, D2[None], c1[None])[0][0] \
        - grad_PQ(mol, c1[None], c2[None])[0][0]
    K = np.array([[np.sum(I[A] * (D1 @ I[B] @ D2)) for B in range(n)] for A in range(n)])
    N = Minv @ K @ Minv
    X1 = [D1 @ I[B] @ D2 for B in range(n)]
    X2 = [D1.T @ I[B] @ D2.T for B in range(n)]
    G = np.stack([sum(Minv[A, B] * (X1[B] + X2[B]) for B in range(n)) for A in range(n)])
    gK = grad_dense_K(mol, G) - grad_PQ_full(mol, N[None])[0]
    return gJ - c_x * gK


# ------------------------------------------------------------------------------------------------
# NEXT-3 / NEXT-4c: products of the ris coupling matrix with trial vectors -- the excitation-energy stage
# (Casida / TDA, Eqs. 1-5 with the ris integrals of Eqs. 20-22) and the ris-approximated
# (A + B) of the Z-vector equation (Eq. 19; Sec. 4.2).  With i, j occupied and a, b virtual,
# Eqs. 2-5 and 20-21 give (the orbital-energy diagonal of A is the caller's)
#   K_{ai,bj} = g^ris_{ai,jb} = (ai|jb)^ris - c_x (ab|ji)^ris        (coupling part of A, Eq. 2)
#   K_{ai,jb} = g^ris_{ai,bj} = (ai|bj)^ris - c_x (aj|bi)^ris        (B, Eq. 3)
#   (pq|sr)^ris = sum_AB (pq|A) M^-1_AB (B|sr)                        (Eq. 21; Coulomb term with the J-fit set and its metric,
#                                                                      exchange terms with the default s set)
# so every product the solvers need is one linear combination
#   sigma_ia = sum_jb [ cJ (ia|jb)^ris - cKA (ij|ab)^ris - cKB (ib|ja)^ris ] X_jb :
#   A-coupling: (1, c_x, 0);  B: (1, 0, c_x);  A + B: (2, c_x, c_x);  A - B: (0, c_x, -c_x)
# (spin-adaptation factors, e.g. cJ = 2 for closed-shell singlets, are the caller's: reading R-sign).
# Tiny molecules only: dense AO tensors, the four-index matrix written out.
def int3c_J(mol, f, *, prim_cutoff=0.0):
    """(mu nu|f) for function f of the J-fit set (the default set when the molecule has none)."""
    h = _Held(mol, jfit=True)
    out = np.zeros((h.nao, h.nao))
    rc = lib().ris_oracle_int3c_P(C.byref(h.c), int(f), prim_cutoff, out.ctypes.data)
    assert rc == 0
    return out


def mo_tensor(I, C_left, C_right):
    """T[P][l][r] = sum_{mu nu} C_left[mu,l] I[P][mu][nu] C_right[nu,r]"""
    return np.einsum("ml,pmn,nr->plr", _f64(C_left), I, _f64(C_right))


def coupling_ris(mol, C_occ, C_vir, cJ, cKA, cKB):
    """The matrix K[i,a,j,b] = cJ (ia|jb)^ris - cKA (ij|ab)^ris - cKB (ib|ja)^ris."""
    nK = np.asarray(mol.coords).shape[0]
    IK = np.stack([int3c(mol, P) for P in range(nK)])
    MJ = metric_J(mol)
    IJ = np.stack([int3c_J(mol, f) for f in range(MJ.shape[0])])
    MJinv, MKinv = np.linalg.inv(MJ), np.linalg.inv(metric(mol))
    Tov_J = mo_tensor(IJ, C_occ, C_vir)
    Too, Tov, Tvv = mo_tensor(IK, C_occ, C_occ), mo_tensor(IK, C_occ, C_vir), mo_tensor(IK, C_vir, C_vir)
    K = cJ * np.einsum("Aia,AB,Bjb->iajb", Tov_J, MJinv, Tov_J)
    K -= cKA * np.einsum("Aij,AB,Bab->iajb", Too, MKinv, Tvv)
    K -= cKB * np.einsum("Aib,AB,Bja->iajb", Tov, MKinv, Tov)
    return K


def matvec_ris(mol, C_occ, C_vir, X, cJ, cKA, cKB):
    """sigma[v][i][a] = sum_jb K[i,a,j,b] X[v][j][b]"""
    return np.einsum("iajb,vjb->via", coupling_ris(mol, C_occ, C_vir, cJ, cKA, cKB), _f64(X))


# --------------------------------------------------------------------------- spherical-harmonic shells (NEXT-4b)
# PAPER.md:170 runs def2-TZVP, a spherical-harmonic basis; SURVEY.md 8(f) NEXT-4 lists the shells, reading R-sph
# fixes the convention: a spherical shell of degree l holds the 2l+1 functions
#     chi_{lm}(r) = S_lm(r - A) sum_k d_k exp(-a_k |r - A|^2),     m = -l .. l  (in this order),
# S_lm the REAL regular solid harmonic in Racah normalisation, S_lm = sqrt(4 pi/(2l+1)) r^l Y_lm^{real}
# (S_00 = 1, S_1m = y, z, x, S_20 = z^2 - (x^2 + y^2)/2, ...).  Its expansion in Cartesian monomials is written out
# from the closed formula (Helgaker, Jorgensen, Olsen, "Molecular Electronic-Structure Theory", Eqs. 6.4.47-6.4.50):
#     S_lm = N_lm sum_{t=0}^{[(l-|m|)/2]} sum_{u=0}^{t} sum_{v} C^{lm}_{tuv} x^{2t+|m|-2(u+v)} y^{2(u+v)} z^{l-2t-|m|},
#     v = v_m, v_m + 1, ..., [|m|/2 - v_m] + v_m,   v_m = 0 (m >= 0) or 1/2 (m < 0),
#     C^{lm}_{tuv} = (-1)^{t+v-v_m} (1/4)^t binom(l,t) binom(l-t,|m|+t) binom(t,u) binom(|m|,2v),
#     N_lm = 1/(2^{|m|} l!) sqrt(2 (l+|m|)! (l-|m|)! / 2^{delta_{m0}}).
# Every integral over spherical functions is the same linear combination of the Cartesian ones, so the contractions in the
# spherical AO basis are the Cartesian ones with D_cart = U^T D_sph U, C_cart = U^T C_sph (U block diagonal).

def _cart_comps(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def solid_harmonic_cart(l: int) -> np.ndarray:
    """T[m + l][c]: coefficient of the Cartesian monomial c (order lx descending, then ly descending) in S_lm."""
    from math import comb, factorial, sqrt
    comps = _cart_comps(l)
    T = np.zeros((2 * l + 1, len(comps)))
    for m in range(-l, l + 1):
        am = abs(m)
        N = sqrt(2.0 * factorial(l + am) * factorial(l - am) / (2.0 if m == 0 else 1.0)) / (2.0 ** am * factorial(l))
        twovm = 0 if m >= 0 else 1                    # 2 v_m
        for t in range((l - am) // 2 + 1):
            for u in range(t + 1):
                # v = v_m + k, k = 0 .. floor(|m|/2 - v_m)
                kmax = (am - twovm) // 2
                for k in range(kmax + 1):
                    twov = twovm + 2 * k              # 2 v  (an odd number for m < 0)
                    sign = (-1) ** (t + k)            # t + v - v_m = t + k
                    Cc = sign * 0.25 ** t * comb(l, t) * comb(l - t, am + t) * comb(t, u) * comb(am, twov)
                    ex = 2 * t + am - 2 * u - twov    # 2t + |m| - 2(u + v)
                    ey = 2 * u + twov                 # 2(u + v)
                    ez = l - 2 * t - am
                    T[m + l, comps.index((ex, ey, ez))] += N * Cc
    return T


def nao_sph(mol) -> int:
    return int(sum(2 * int(l) + 1 for l in mol.shell_l))


def sph_matrix(mol) -> np.ndarray:
    """U[nao_sph][nao_cart], block diagonal over the shells: chi^sph = U chi^cart."""
    ls = [int(l) for l in mol.shell_l]
    U = np.zeros((sum(2 * l + 1 for l in ls), sum((l + 1) * (l + 2) // 2 for l in ls)))
    r = c = 0
    for l in ls:
        T = solid_harmonic_cart(l)
        U[r:r + T.shape[0], c:c + T.shape[1]] = T
        r += T.shape[0]; c += T.shape[1]
    return U


def density_sph_to_cart(mol, D_sph):
    """D_cart = U^T D_sph U for [nbatch][nao_sph][nao_sph] (or one matrix)."""
    U = sph_matrix(mol)
    return U.T @ _f64(D_sph) @ U          # matmul broadcasts over the leading state index


def coef_sph_to_cart(mol, C_sph):
    """C_cart = U^T C_sph for [nao_sph][n]."""
    return sph_matrix(mol).T @ _f64(C_sph)


def grad_J_sph(mol, D_sph, c_aux, **kw):
    return grad_J(mol, density_sph_to_cart(mol, D_sph), c_aux, **kw)


def grad_K_sph(mol, C_occ_sph, C_vir_sph, B, **kw):
    return grad_K(mol, coef_sph_to_cart(mol, C_occ_sph), coef_sph_to_cart(mol, C_vir_sph), B, **kw)


def int3c_sph(mol, P, **kw):
    """(mu nu|P) over the spherical functions of the molecule, [nao_sph][nao_sph]."""
    U = sph_matrix(mol)
    return U @ int3c(mol, P, **kw) @ U.T
