"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each checks the oracle against something other than
itself: printed reference values (tests/golden/), closed forms, mpmath special functions,
brute-force quadrature, finite differences, invariances.
"""
import itertools
import math
import os

import mpmath
import numpy as np
import pytest

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")
A0 = np.array([0.1, -0.3, 0.2])
B0 = np.array([0.9, 0.4, -0.5])
C0 = np.array([-0.7, 1.1, 0.6])


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------ P3: Boys function

def test_boys_golden_values():
    for T, m, ref in _rows("boys_reference.txt"):
        got = orc.boys(8, float(T))[int(m)]
        assert abs(got - float(ref)) <= 2e-15 * abs(float(ref))


def test_boys_zero_argument():
    F = orc.boys(9, 0.0)
    for m in range(10):
        assert abs(F[m] - 1.0 / (2 * m + 1)) < 1e-16


@pytest.mark.parametrize("T", [1e-9, 1e-3, 0.5, 5.0, 20.0, 25.0, 33.0, 34.999, 35.0, 50.0, 100.0, 1e3, 1e5])
def test_boys_incomplete_gamma(T):
    """F_m(T) = gamma(m+1/2, T) / (2 T^(m+1/2)) in 40-digit arithmetic."""
    mpmath.mp.dps = 40
    F = orc.boys(9, T)
    for m in range(10):
        ref = mpmath.gammainc(m + 0.5, 0, T) / (2 * mpmath.mpf(T) ** (m + 0.5))
        assert abs(F[m] - float(ref)) <= 4e-15 * float(ref), (T, m)


def test_boys_quadrature_of_definition():
    x, w = np.polynomial.legendre.leggauss(200)
    t = 0.5 * (x + 1.0)
    for T in (0.3, 7.0, 31.0, 60.0):
        F = orc.boys(6, T)
        for m in range(7):
            ref = 0.5 * np.sum(w * t ** (2 * m) * np.exp(-T * t * t))
            assert abs(F[m] - ref) <= 1e-13 * ref


def test_boys_erf_closed_form():
    for T in (0.2, 3.0, 36.0, 80.0):
        assert abs(orc.boys(0, T)[0] - 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))) < 1e-15


# ------------------------------------------------------------------ P1/P2: closed-form s-s-s

def _sss_closed(a, b, alpha, A, B, Cc):
    p = a + b
    rho = p * alpha / (p + alpha)
    P = (a * A + b * B) / p
    Kab = math.exp(-a * b / p * np.dot(A - B, A - B))
    kappa = 2 * math.pi ** 2.5 / (p * alpha * math.sqrt(p + alpha)) * Kab
    T = rho * np.dot(P - Cc, P - Cc)
    mpmath.mp.dps = 30
    F0 = float(mpmath.gammainc(0.5, 0, T) / (2 * mpmath.sqrt(T))) if T > 0 else 1.0
    F1 = float(mpmath.gammainc(1.5, 0, T) / (2 * mpmath.mpf(T) ** 1.5)) if T > 0 else 1.0 / 3
    val = kappa * F0
    dA = kappa * (-2 * (a * b / p) * (A - B) * F0 - 2 * rho * (a / p) * (P - Cc) * F1)
    dB = kappa * (-2 * (a * b / p) * (B - A) * F0 - 2 * rho * (b / p) * (P - Cc) * F1)
    dC = 2 * rho * (P - Cc) * kappa * F1
    return val, dA, dB, dC


@pytest.mark.parametrize("seed", range(6))
def test_sss_closed_form_value_and_gradient(seed):
    rng = np.random.default_rng(100 + seed)
    a, b, alpha = np.exp(rng.uniform(-2, 3, 3))
    A, B, Cc = rng.normal(size=(3, 3)) * (0.5 + 2 * seed)
    val, dA, dB, dC = _sss_closed(a, b, alpha, A, B, Cc)
    got = orc.prim3c((0, 0, 0), (0, 0, 0), a, b, alpha, A, B, Cc)
    scale = abs(val)
    assert abs(got[0] - val) <= 1e-14 * scale
    np.testing.assert_allclose(got[1:4], dA, rtol=0, atol=2e-14 * max(scale, np.abs(dA).max()))
    np.testing.assert_allclose(got[4:7], dB, rtol=0, atol=2e-14 * max(scale, np.abs(dB).max()))
    np.testing.assert_allclose(got[7:10], dC, rtol=0, atol=2e-14 * max(scale, np.abs(dC).max()))


def test_sss_aux_on_product_centre_T_zero():
    a, b, alpha = 0.7, 0.7, 0.3
    A, B = np.array([0.0, 0, 1.0]), np.array([0.0, 0, -1.0])
    Cc = np.zeros(3)       # = P, so T = 0
    val, dA, dB, dC = _sss_closed(a, b, alpha, A, B, Cc)
    got = orc.prim3c((0, 0, 0), (0, 0, 0), a, b, alpha, A, B, Cc)
    assert abs(got[0] - val) < 1e-14 * val
    np.testing.assert_allclose(got[1:4], dA, atol=1e-14 * val)
    np.testing.assert_allclose(got[7:10], 0.0, atol=1e-15)


# ------------------------------------------------------------------ P4/P5: worked example

def test_worked_example_three_centre():
    rows = _rows("prim3c_worked_example.txt")
    for r in rows:
        if r[0] == "grad":
            ref = np.array([float(x) for x in r[1:]])
            got = orc.prim3c((0, 0, 0), (0, 0, 0), 0.8, 1.3, 0.25, A0, B0, C0)[1:]
            np.testing.assert_allclose(got, ref, rtol=1e-13)
        else:
            la, lb, ref = tuple(map(int, r[0:3])), tuple(map(int, r[3:6])), float(r[6])
            got = orc.prim3c(la, lb, 0.8, 1.3, 0.25, A0, B0, C0)[0]
            assert abs(got - ref) <= 1e-13 * abs(ref)


def test_worked_example_two_centre():
    ref = np.array([float(x) for x in _rows("prim2c_worked_example.txt")[0]])
    got = orc.prim2c(0.3, 0.7, C0, A0)
    np.testing.assert_allclose(got, ref, rtol=1e-13)


def test_two_centre_closed_form_and_antisymmetry():
    mpmath.mp.dps = 30
    rng = np.random.default_rng(7)
    for _ in range(5):
        al, be = np.exp(rng.uniform(-3, 1, 2))
        RP, RQ = rng.normal(size=(2, 3)) * 3
        rho = al * be / (al + be)
        T = rho * np.dot(RP - RQ, RP - RQ)
        pref = 2 * math.pi ** 2.5 / (al * be * math.sqrt(al + be))
        F0 = float(mpmath.gammainc(0.5, 0, T) / (2 * mpmath.sqrt(T)))
        F1 = float(mpmath.gammainc(1.5, 0, T) / (2 * mpmath.mpf(T) ** 1.5))
        got = orc.prim2c(al, be, RP, RQ)
        assert abs(got[0] - pref * F0) < 1e-14 * pref * F0
        np.testing.assert_allclose(got[1:], -2 * rho * (RP - RQ) * pref * F1, rtol=1e-13)
        swapped = orc.prim2c(be, al, RQ, RP)
        np.testing.assert_allclose(swapped[1:], -got[1:], rtol=1e-13)
    # coincident centres: finite value, zero derivative
    got = orc.prim2c(0.4, 0.9, RP, RP)
    assert abs(got[0] - 2 * math.pi ** 2.5 / (0.36 * math.sqrt(1.3))) < 1e-12
    assert np.all(got[1:] == 0.0)


# ------------------------------------------------------------------ P8: brute-force quadrature

def _quad3c(la, lb, a, b, alpha, A, B, Cc, n=48):
    """int phi_a(r) phi_b(r) V_C(r) dr by 3-D Gauss-Hermite on the product Gaussian.
    V_C(r) = (pi/alpha)^(3/2) erf(sqrt(alpha)|r-C|)/|r-C| is the potential of exp(-alpha|r-C|^2)."""
    from scipy.special import erf
    p = a + b
    P = (a * A + b * B) / p
    Kab = math.exp(-a * b / p * np.dot(A - B, A - B))
    x, w = np.polynomial.hermite.hermgauss(n)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    W = w[:, None, None] * w[None, :, None] * w[None, None, :]
    r = np.stack([X, Y, Z], -1) / math.sqrt(p) + P
    poly = np.ones_like(X)
    for d in range(3):
        poly = poly * (r[..., d] - A[d]) ** la[d] * (r[..., d] - B[d]) ** lb[d]
    dist = np.linalg.norm(r - Cc, axis=-1)
    V = (math.pi / alpha) ** 1.5 * erf(math.sqrt(alpha) * dist) / dist
    return Kab * p ** -1.5 * np.sum(W * poly * V)


def _comps(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


@pytest.mark.parametrize("la,lb", [(0, 0), (1, 0), (1, 1), (2, 0), (2, 1), (2, 2), (3, 1), (3, 3)])
def test_quadrature_values_per_class(la, lb):
    a, b, alpha = 0.9, 0.6, 0.35
    A, B, Cc = np.array([0.2, -0.1, 0.3]), np.array([-0.4, 0.5, 0.1]), np.array([1.9, -1.4, 1.1])
    ca, cb = _comps(la), _comps(lb)
    picks = [(ca[0], cb[0]), (ca[-1], cb[-1]), (ca[len(ca) // 2], cb[len(cb) // 2]), (ca[-1], cb[0])]
    for xa, xb in picks:
        got = orc.prim3c(xa, xb, a, b, alpha, A, B, Cc)[0]
        ref = _quad3c(xa, xb, a, b, alpha, A, B, Cc)
        assert abs(got - ref) <= 2e-11 * max(1.0, abs(ref)), (xa, xb, got, ref)


def test_quadrature_finite_difference_of_derivatives():
    """All nine derivative numbers of a d-p primitive vs central differences of the quadrature."""
    a, b, alpha = 0.9, 0.6, 0.35
    A, B, Cc = np.array([0.2, -0.1, 0.3]), np.array([-0.4, 0.5, 0.1]), np.array([1.9, -1.4, 1.1])
    xa, xb = (1, 0, 1), (0, 1, 0)
    got = orc.prim3c(xa, xb, a, b, alpha, A, B, Cc)
    h = 1e-4
    for which, base in enumerate((A, B, Cc)):
        for d in range(3):
            args_p, args_m = [A.copy(), B.copy(), Cc.copy()], [A.copy(), B.copy(), Cc.copy()]
            args_p[which][d] += h
            args_m[which][d] -= h
            fd = (_quad3c(xa, xb, a, b, alpha, *args_p, n=40) - _quad3c(xa, xb, a, b, alpha, *args_m, n=40)) / (2 * h)
            assert abs(got[1 + 3 * which + d] - fd) < 1e-6, (which, d)


def test_quadrature_finite_difference_of_f_shell_derivatives():
    """l = 3 in the differentiated function: all nine derivative numbers of an f-d primitive pair (the `2a[a+1|`
    branch with l_a + 1 = 4: E table index 4, Hermite R order 8; Eq. 27 terms 1-2) vs central
    differences of the brute-force quadrature.  Two component pairs so that every Cartesian direction is raised to 4."""
    a, b, alpha = 0.9, 0.6, 0.35
    A, B, Cc = np.array([0.2, -0.1, 0.3]), np.array([-0.4, 0.5, 0.1]), np.array([1.9, -1.4, 1.1])
    h = 1e-4
    for xa, xb in (((3, 0, 0), (0, 1, 1)), ((0, 2, 1), (1, 0, 1)), ((0, 0, 3), (0, 2, 0))):
        got = orc.prim3c(xa, xb, a, b, alpha, A, B, Cc)
        scale = max(1.0, np.abs(got[1:]).max())
        for which in range(3):
            for d in range(3):
                args_p, args_m = [A.copy(), B.copy(), Cc.copy()], [A.copy(), B.copy(), Cc.copy()]
                args_p[which][d] += h
                args_m[which][d] -= h
                fd = (_quad3c(xa, xb, a, b, alpha, *args_p, n=44) - _quad3c(xa, xb, a, b, alpha, *args_m, n=44)) / (2 * h)
                assert abs(got[1 + 3 * which + d] - fd) < 2e-6 * scale, (xa, xb, which, d, got[1 + 3 * which + d], fd)


# ------------------------------------------------------------------ P12: far-aux limit

def test_far_aux_limit():
    """(ss|P) -> S_ab (pi/alpha)^(3/2) / R for a far auxiliary centre (exact for s-s: both charge clouds
    are spherical about P and C)."""
    a, b, alpha = 1.1, 0.4, 0.2
    A, B = np.array([0.0, 0.3, 0.0]), np.array([0.5, 0.0, -0.2])
    Cc = np.array([200.0, 0.0, 0.0])
    p = a + b
    P = (a * A + b * B) / p
    S = (math.pi / p) ** 1.5 * math.exp(-a * b / p * np.dot(A - B, A - B))
    ref = S * (math.pi / alpha) ** 1.5 / np.linalg.norm(P - Cc)
    got = orc.prim3c((0, 0, 0), (0, 0, 0), a, b, alpha, A, B, Cc)[0]
    assert abs(got - ref) < 1e-13 * ref
    # p-s product: monopole S_ab-like term plus a dipole ~ 1/R^2 -> agreement ~1/R
    got = orc.prim3c((1, 0, 0), (0, 0, 0), a, b, alpha, A, B, Cc)[0]
    mono = S * (P[0] - A[0]) * (math.pi / alpha) ** 1.5 / np.linalg.norm(P - Cc)
    assert abs(got - mono) < 2e-2 * abs(mono)


# ------------------------------------------------------------------ contraction-level pins

def _wl1():
    return synth.make_workload(1)


def _small():
    """3 atoms, spd shells, two primitives each: a fast stand-in with every class up to (2,2)."""
    mol = synth.tiny_molecule(5, [[0, 1, 2], [0, 1], [2, 0]],
                              [[0.0, 0.0, 0.0], [1.6, 0.3, -0.2], [-0.7, 1.5, 0.9]])
    rng = np.random.default_rng(11)
    nao = mol.nao
    return mol, rng.standard_normal((2, nao, nao)), rng.standard_normal((2, 3)), rng


def _displaced(mol, atom, d, h):
    import copy
    m2 = copy.copy(mol)
    m2.coords = mol.coords.copy()
    m2.coords[atom, d] += h
    return m2


def test_finite_difference_config1_all_atoms():
    """P6 (PAPER.md:702-704 validates the same way): central differences, step 5e-6 bohr, of E_J, E_K and
    E_PQ at fixed D, c, C, B, for every atom and direction of config 1."""
    wl = _wl1()
    mol = wl.mol
    gJ, _ = orc.grad_J(mol, wl.D, wl.c_aux)
    gK, _ = orc.grad_K(mol, wl.C_occ, wl.C_vir, wl.B)
    gQ, _ = orc.grad_PQ(mol, wl.c_aux, wl.d_aux)
    h = 5e-6
    for atom, d in itertools.product(range(3), range(3)):
        mp_, mm_ = _displaced(mol, atom, d, h), _displaced(mol, atom, d, -h)
        for name, g, f in (("J", gJ, lambda m: orc.grad_J(m, wl.D, wl.c_aux)[1]),
                           ("K", gK, lambda m: orc.grad_K(m, wl.C_occ, wl.C_vir, wl.B)[1]),
                           ("PQ", gQ, lambda m: orc.grad_PQ(m, wl.c_aux, wl.d_aux)[1])):
            fd = (f(mp_)[0] - f(mm_)[0]) / (2 * h)
            scale = np.abs(g[0]).max()
            assert abs(g[0, atom, d] - fd) < 2e-7 * scale, (name, atom, d, g[0, atom, d], fd)


def test_finite_difference_f_shells_all_atoms():
    """P6 at l = 3: central differences (5e-6 bohr) of E_J and E_K for every atom and direction of a
    3-atom molecule with shells [[f, s], [f, d], [p]] -- classes (3,3), (3,2), (3,1), (3,0) differentiate an f shell, i.e.
    the oracle's table bounds EMAX = 4 / Hermite order 8 are exercised without the CUDA path vouching for them."""
    mol = synth.tiny_molecule(31, [[3, 0], [3, 2], [1]], [[0.0, 0.0, 0.0], [1.7, 0.4, -0.3], [-0.6, 1.6, 0.8]])
    rng = np.random.default_rng(32)
    nao, nocc, nvir = mol.nao, 3, 4
    D = rng.standard_normal((1, nao, nao))
    c = rng.standard_normal((1, 3))
    Co, Cv = rng.standard_normal((nao, nocc)), rng.standard_normal((nao, nvir))
    B = rng.standard_normal((1, 3, nocc, nvir))
    gJ, _ = orc.grad_J(mol, D, c)
    gK, _ = orc.grad_K(mol, Co, Cv, B)
    assert np.all(np.abs(gJ.sum(axis=1)) < 1e-12 * np.abs(gJ).sum())
    assert np.all(np.abs(gK.sum(axis=1)) < 1e-12 * np.abs(gK).sum())
    h = 5e-6
    for atom, d in itertools.product(range(3), range(3)):
        mp_, mm_ = _displaced(mol, atom, d, h), _displaced(mol, atom, d, -h)
        for name, g, f in (("J", gJ, lambda m: orc.grad_J(m, D, c)[1]), ("K", gK, lambda m: orc.grad_K(m, Co, Cv, B)[1])):
            fd = (f(mp_)[0] - f(mm_)[0]) / (2 * h)
            assert abs(g[0, atom, d] - fd) < 2e-7 * np.abs(g[0]).max(), (name, atom, d, g[0, atom, d], fd)


def test_finite_difference_directional_all_classes():
    """Directional derivative along random collective displacements on a molecule with d shells on
    two atoms (classes up to (2,2), two states at once)."""
    mol, D, c, rng = _small()
    g, _ = orc.grad_J(mol, D, c)
    h = 5e-6
    for _ in range(3):
        v = rng.standard_normal(mol.coords.shape)
        import copy
        mp_, mm_ = copy.copy(mol), copy.copy(mol)
        mp_.coords = mol.coords + h * v
        mm_.coords = mol.coords - h * v
        fd = (orc.grad_J(mp_, D, c)[1] - orc.grad_J(mm_, D, c)[1]) / (2 * h)
        an = np.einsum("sax,ax->s", g, v)
        assert np.all(np.abs(an - fd) < 2e-7 * np.abs(g).max() * np.abs(v).sum())


def test_translational_invariance_each_term():
    """P7: each of J, K, PQ sums to zero over atoms (north_star: 1e-10 relative)."""
    wl = _wl1()
    for g in (orc.grad_J(wl.mol, wl.D, wl.c_aux)[0], orc.grad_K(wl.mol, wl.C_occ, wl.C_vir, wl.B)[0],
              orc.grad_PQ(wl.mol, wl.c_aux, wl.d_aux)[0]):
        assert np.all(np.abs(g.sum(axis=1)) < 1e-10 * np.abs(g).sum())


def test_symmetry_linearity_batch_independence():
    """P9."""
    mol, D, c, rng = _small()
    g, e = orc.grad_J(mol, D, c)
    gT, _ = orc.grad_J(mol, D.transpose(0, 2, 1), c)
    np.testing.assert_allclose(gT, g, rtol=0, atol=1e-13 * np.abs(g).max())
    gsym, _ = orc.grad_J(mol, 0.5 * (D + D.transpose(0, 2, 1)), c)
    np.testing.assert_allclose(gsym, g, rtol=0, atol=1e-13 * np.abs(g).max())
    g0, _ = orc.grad_J(mol, D[:1], c[:1])            # batch entries are independent
    np.testing.assert_allclose(g0[0], g[0], rtol=0, atol=1e-13 * np.abs(g).max())
    glin, _ = orc.grad_J(mol, 2.0 * D[0] - 3.0 * D[1], c[:1])
    gb, _ = orc.grad_J(mol, D[1], c[:1])
    np.testing.assert_allclose(glin[0], 2.0 * g[0] - 3.0 * gb[0], rtol=0, atol=1e-12 * np.abs(g).max())


def test_K_reduces_to_J():
    """P10: D = C_occ X C_vir^T, B[P] = c_P X  =>  grad_K = grad_J(D, c)."""
    mol, _, c, rng = _small()
    nocc, nvir = 3, 4
    Co, Cv = rng.standard_normal((mol.nao, nocc)), rng.standard_normal((mol.nao, nvir))
    X = rng.standard_normal((nocc, nvir))
    B = c[0][:, None, None] * X[None]
    gK, eK = orc.grad_K(mol, Co, Cv, B[None])
    gJ, eJ = orc.grad_J(mol, (Co @ X @ Cv.T)[None], c[:1])
    np.testing.assert_allclose(gK, gJ, rtol=0, atol=1e-12 * np.abs(gJ).max())
    assert abs(eK[0] - eJ[0]) < 1e-12 * abs(eJ[0])


def test_permutation_of_atoms_and_shells():
    """P11: relabelling atoms / reordering shells permutes the result."""
    mol, D, c, rng = _small()
    g, _ = orc.grad_J(mol, D[:1], c[:1])
    perm = np.array([2, 0, 1])                        # new atom k = old atom perm[k]
    inv = np.argsort(perm)
    sh = np.array([4, 0, 6, 2, 5, 1, 3])              # new shell k = old shell sh[k]
    import copy
    m2 = copy.copy(mol)
    m2.coords = mol.coords[perm]
    m2.aux_exponents = mol.aux_exponents[perm]
    m2.shell_atom = inv[mol.shell_atom[sh]].astype(np.int32)
    m2.shell_l = mol.shell_l[sh]
    m2.shell_nprim = mol.shell_nprim[sh]
    m2.shell_prim_off = mol.shell_prim_off[sh]
    off = mol.ao_off
    aoperm = np.concatenate([np.arange(off[s], off[s] + synth.ncart(int(mol.shell_l[s]))) for s in sh])
    D2 = D[:1][:, aoperm][:, :, aoperm]
    g2, _ = orc.grad_J(m2, D2, c[:1][:, perm])
    np.testing.assert_allclose(g2[0], g[0][perm], rtol=0, atol=1e-12 * np.abs(g).max())


def test_single_atom_is_exactly_zero_and_s_only_has_no_torque():
    mol = synth.tiny_molecule(3, [[0, 1, 2]], [[0.3, -0.2, 0.5]])
    rng = np.random.default_rng(0)
    g, _ = orc.grad_J(mol, rng.standard_normal((1, mol.nao, mol.nao)), rng.standard_normal((1, 1)))
    assert np.abs(g).max() < 1e-13        # three centres on one atom: dA + dB + dC = 0
    mol = synth.tiny_molecule(4, [[0, 0], [0], [0, 0]], [[0.0, 0, 0], [1.5, 0.2, 0.1], [0.3, 1.4, -0.8]])
    D = rng.standard_normal((1, mol.nao, mol.nao))
    g, _ = orc.grad_J(mol, D, rng.standard_normal((1, 3)))
    torque = np.cross(mol.coords, g[0]).sum(axis=0)
    assert np.abs(torque).max() < 1e-12 * np.abs(g).max()


def test_sampled_atoms_and_cutoff_equal_full():
    """The `atoms=` sampling and the documented 1e-22 primitive cutoff reproduce the
    unrestricted definition."""
    wl = synth.make_workload(1)
    gJ, _ = orc.grad_J(wl.mol, wl.D, wl.c_aux)
    gK, _ = orc.grad_K(wl.mol, wl.C_occ, wl.C_vir, wl.B)
    for atoms in ([0], [2], [1, 2]):
        sJ, _ = orc.grad_J(wl.mol, wl.D, wl.c_aux, atoms=atoms)
        sK, _ = orc.grad_K(wl.mol, wl.C_occ, wl.C_vir, wl.B, atoms=atoms)
        np.testing.assert_allclose(sJ[:, atoms], gJ[:, atoms], rtol=0, atol=1e-13 * np.abs(gJ).max())
        np.testing.assert_allclose(sK[:, atoms], gK[:, atoms], rtol=0, atol=1e-13 * np.abs(gK).max())
        others = [a for a in range(3) if a not in atoms]
        assert np.all(np.isnan(sJ[:, others]))
    cJ, _ = orc.grad_J(wl.mol, wl.D, wl.c_aux, prim_cutoff=1e-22)
    np.testing.assert_allclose(cJ, gJ, rtol=0, atol=1e-14 * np.abs(gJ).max())


# ------------------------------------------------------------------ the oracle's own FP64 rounding error (R-tol evidence)

@pytest.mark.parametrize("cfg", [1, 2])
def test_fp64_oracle_against_its_extended_precision_build(cfg):
    """DESIGN.md reading R-tol rests on this measurement: the oracle (FP64 intermediates) against the SAME source built
    with every intermediate in `long double` (-DORACLE_REAL, 64-bit mantissa) differs by a few 1e-15 of the gradient's
    largest component -- so `5e-14 * max|ref|` (tests/test_gpu_parity.py) is ~30x the oracle's own rounding noise, and an
    absolute floor has to be expressed in units of the gradient.  Also: against the extended build the FP64 oracle passes
    north_star's LITERAL tolerance 1e-12 + 1e-10 |ref| on every component."""
    wl = synth.make_workload(cfg)
    mol = wl.mol
    ref64 = (orc.grad_J(mol, wl.D, wl.c_aux)[0], orc.grad_K(mol, wl.C_occ, wl.C_vir, wl.B)[0],
             orc.grad_PQ(mol, wl.c_aux, wl.d_aux)[0])
    with orc.extended_precision():
        ext = (orc.grad_J(mol, wl.D, wl.c_aux)[0], orc.grad_K(mol, wl.C_occ, wl.C_vir, wl.B)[0],
               orc.grad_PQ(mol, wl.c_aux, wl.d_aux)[0])
    again = orc.grad_J(mol, wl.D, wl.c_aux)[0]
    # the context manager restored the FP64 build (OpenMP merges the threads' long double partial sums in arrival
    # order, so two runs agree to the last bit or so, not necessarily bitwise)
    assert np.abs(again - ref64[0]).max() <= 3e-16 * np.abs(again).max()
    # measured: config 1  J 1.4e-14 (tight same-atom pairs, exponent ratio up to 500), K 2.4e-15, PQ 1.9e-16;
    #           config 2  J 1.7e-15, K 1.6e-15, PQ 2.0e-16
    bound = {1: 3e-14, 2: 5e-15}[cfg]
    for name, a, b in zip("J K PQ".split(), ref64, ext):
        err = np.abs(a - b)
        assert err.max() <= bound * np.abs(b).max(), (name, err.max() / np.abs(b).max())
        assert np.all(err <= 1e-12 + 1e-10 * np.abs(b)), (name, (err / (1e-12 + 1e-10 * np.abs(b))).max())
