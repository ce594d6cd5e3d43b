"""Pins of the oracle's p-type auxiliary functions ("a single GTO for each angular
momentum component (up to l = 2) on each atom"; "s- and p-type for Coulomb, only s-type for exchange").

None of these touches the CUDA path.  Each checks the oracle against something other than itself: brute-force quadrature
with the closed-form potential of a p-type Gaussian charge, the identity p_i = (1/2 alpha) d/dC_i s applied to the
ALREADY PINNED s-type integrals, closed forms in Boys functions evaluated by mpmath, finite differences through the
metric solve, invariances."""
import copy
import itertools
import math

import mpmath
import numpy as np
import pytest

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import synth


def _comps(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def _quad3c_p(la, lb, a, b, alpha, A, B, Cc, i, n=48):
    """int phi_a phi_b V_i dr by 3-D Gauss-Hermite; V_i = potential of the UNNORMALISED p primitive (r-C)_i e^{-alpha|r-C|^2}
    = (1/2 alpha) d/dC_i [(pi/alpha)^{3/2} erf(sqrt(alpha) d)/d],  d = |r - C|:
      d/dC_i f(d) = -f'(d) (r-C)_i / d,   f = erf(sqrt(alpha) d)/d,  f' = (2 sqrt(alpha/pi) e^{-alpha d^2} d - erf(sqrt(alpha) d))/d^2."""
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
    sa = math.sqrt(alpha)
    fp = (2 * sa / math.sqrt(math.pi) * np.exp(-alpha * dist ** 2) * dist - erf(sa * dist)) / dist ** 2
    V = (math.pi / alpha) ** 1.5 / (2 * alpha) * (-fp) * (r[..., i] - Cc[i]) / dist
    return Kab * p ** -1.5 * np.sum(W * poly * V)


GEOM = (np.array([0.2, -0.1, 0.3]), np.array([-0.4, 0.5, 0.1]), np.array([1.9, -1.4, 1.1]))


@pytest.mark.parametrize("la,lb", [(0, 0), (1, 0), (1, 1), (2, 0), (2, 1), (2, 2), (3, 1)])
def test_p_aux_values_against_quadrature(la, lb):
    a, b, alpha = 0.9, 0.6, 0.35
    A, B, Cc = GEOM
    ca, cb = _comps(la), _comps(lb)
    for (xa, xb), i in zip([(ca[0], cb[0]), (ca[-1], cb[-1]), (ca[len(ca) // 2], cb[len(cb) // 2])], (0, 1, 2)):
        got = orc.prim3c_aux(xa, xb, a, b, alpha, A, B, Cc, 1, i)[0]
        ref = _quad3c_p(xa, xb, a, b, alpha, A, B, Cc, i)
        assert abs(got - ref) <= 2e-11 * max(1.0, abs(ref)), (xa, xb, i, got, ref)


@pytest.mark.parametrize("comp", [0, 1, 2])
def test_p_aux_is_the_centre_derivative_of_the_pinned_s_aux(comp):
    """(ab|p_i) = (1/2 alpha) d/dC_i (ab|s): the s-aux oracle returns d/dC analytically (pinned in test_oracle_pins.py), so
    the p-aux VALUE must equal it; and the p-aux DERIVATIVES must equal central differences of that identity."""
    a, b, alpha = 1.3, 0.45, 0.28
    A, B, Cc = GEOM
    for xa, xb in (((0, 0, 0), (0, 0, 0)), ((1, 0, 1), (0, 1, 0)), ((2, 0, 0), (0, 1, 1)), ((0, 3, 0), (1, 0, 1))):
        s = orc.prim3c(xa, xb, a, b, alpha, A, B, Cc)
        p = orc.prim3c_aux(xa, xb, a, b, alpha, A, B, Cc, 1, comp)
        assert abs(p[0] - s[7 + comp] / (2 * alpha)) <= 1e-13 * max(1.0, abs(p[0]))
        h = 1e-4
        for which in range(3):
            for d in range(3):
                args_p, args_m = [A.copy(), B.copy(), Cc.copy()], [A.copy(), B.copy(), Cc.copy()]
                args_p[which][d] += h
                args_m[which][d] -= h
                fd = (orc.prim3c(xa, xb, a, b, alpha, *args_p)[7 + comp] - orc.prim3c(xa, xb, a, b, alpha, *args_m)[7 + comp]) / (2 * h) / (2 * alpha)
                assert abs(p[1 + 3 * which + d] - fd) < 3e-7 * max(1.0, np.abs(p[1:]).max()), (xa, xb, which, d)
        # translational invariance of the primitive: dA + dB + dC = 0
        np.testing.assert_allclose(p[1:4] + p[4:7] + p[7:10], 0.0, atol=1e-13 * max(1.0, np.abs(p[1:]).max()))


def test_two_centre_s_p_and_p_p_closed_forms():
    """(p_i|s) = (1/2 alpha) d/dC_i (s|s) (from the pinned prim2c), (p_i|p_j) = (kappa / 4 alpha beta)(2 rho delta_ij F_1 -
    4 rho^2 X_i X_j F_2) with Boys values from mpmath; derivatives by central differences."""
    mpmath.mp.dps = 30
    rng = np.random.default_rng(5)
    for _ in range(4):
        al, be = np.exp(rng.uniform(-2.5, 0.5, 2))
        RP, RQ = rng.normal(size=(2, 3)) * 2.0
        X = RP - RQ
        rho = al * be / (al + be)
        T = rho * float(X @ X)
        kappa = 2 * math.pi ** 2.5 / (al * be * math.sqrt(al + be))
        F = [float(mpmath.gammainc(m + 0.5, 0, T) / (2 * mpmath.mpf(T) ** (m + 0.5))) for m in range(3)]
        ss = orc.prim2c(al, be, RP, RQ)
        for i in range(3):
            ps = orc.prim2c_lm(al, be, 1, i, 0, 0, RP, RQ)
            assert abs(ps[0] - ss[1 + i] / (2 * al)) <= 1e-13 * abs(ss[0])
            sp = orc.prim2c_lm(al, be, 0, 0, 1, i, RP, RQ)
            assert abs(sp[0] + ss[1 + i] / (2 * be)) <= 1e-13 * abs(ss[0])        # d/dR_Q = -d/dR_P
            for j in range(3):
                pp = orc.prim2c_lm(al, be, 1, i, 1, j, RP, RQ)
                ref = kappa / (4 * al * be) * (2 * rho * (i == j) * F[1] - 4 * rho ** 2 * X[i] * X[j] * F[2])
                assert abs(pp[0] - ref) <= 1e-13 * abs(kappa / (4 * al * be)), (i, j, pp[0], ref)
                h = 1e-4
                for d in range(3):
                    Rp, Rm = RP.copy(), RP.copy()
                    Rp[d] += h; Rm[d] -= h
                    fd = (orc.prim2c_lm(al, be, 1, i, 1, j, Rp, RQ)[0] - orc.prim2c_lm(al, be, 1, i, 1, j, Rm, RQ)[0]) / (2 * h)
                    assert abs(pp[1 + d] - fd) < 1e-6 * abs(kappa / (4 * al * be))


def test_p_function_is_normalised():
    """N_p^2 int x^2 e^{-2 alpha r^2} d^3r = 1 through the metric's diagonal: the self-repulsion of the normalised p function
    has the closed form (p_i|p_i) N_p^2 = N_p^2 kappa 2 rho F_1(0) / (4 alpha^2) = (16/15) ... checked numerically against a
    radial quadrature of the definition instead of a remembered constant."""
    alpha = 0.37
    Np2 = ((2 * alpha / math.pi) ** 0.75 * 2 * math.sqrt(alpha)) ** 2
    x, w = np.polynomial.hermite.hermgauss(40)
    # int x^2 e^{-2 alpha x^2} dx * (int e^{-2 alpha y^2} dy)^2
    s = math.sqrt(2 * alpha)
    ix2 = np.sum(w * (x / s) ** 2) / s
    i0 = np.sum(w) / s
    assert abs(Np2 * ix2 * i0 * i0 - 1.0) < 1e-13
    mol = synth.tiny_molecule(3, [[0]], [[0.0, 0.0, 0.0]])
    mol.jfit = (np.array([0]), np.array([1]), np.array([alpha]))
    M = orc.metric_J(mol)
    # the three components are degenerate and orthogonal; (p|p) self-repulsion > 0
    assert np.allclose(M, np.eye(3) * M[0, 0], atol=1e-14) and M[0, 0] > 0
    # closed form: N_p^2 * kappa/(4 alpha^2) * 2 rho F_1(0), rho = alpha/2, F_1(0) = 1/3
    kappa = 2 * math.pi ** 2.5 / (alpha * alpha * math.sqrt(2 * alpha))
    assert abs(M[0, 0] - Np2 * kappa / (4 * alpha ** 2) * 2 * (alpha / 2) / 3) < 1e-13 * M[0, 0]


# ---------------------------------------------------------------------- contraction level

def _mol_sp():
    """3 atoms, spd shells, one s + one p auxiliary shell per atom (the J-fit set of PAPER.md:168)."""
    mol = synth.tiny_molecule(5, [[0, 1, 2], [0, 1], [2, 0]], [[0.0, 0.0, 0.0], [1.6, 0.3, -0.2], [-0.7, 1.5, 0.9]])
    mol.jfit = (np.array([0, 0, 1, 1, 2, 2]), np.array([0, 1, 0, 1, 0, 1]), np.array([0.31, 0.42, 0.22, 0.53, 0.27, 0.36]))
    return mol


def _displaced(mol, atom, d, h):
    m2 = copy.copy(mol)
    m2.coords = mol.coords.copy()
    m2.coords[atom, d] += h
    return m2


def test_finite_difference_J_and_PQ_with_p_functions():
    """P6 with the s+p J-fit set: central differences (5e-6 bohr) of E_J and E_PQ at fixed D, c for every atom and
    direction; each term sums to zero over the atoms (P7)."""
    mol = _mol_sp()
    rng = np.random.default_rng(12)
    D = rng.standard_normal((1, mol.nao, mol.nao))
    c, dq = rng.standard_normal((2, 1, 12))
    gJ, _ = orc.grad_J(mol, D, c)
    gQ, _ = orc.grad_PQ(mol, c, dq)
    for g in (gJ, gQ):
        assert np.all(np.abs(g.sum(axis=1)) < 1e-12 * np.abs(g).sum())
    h = 5e-6
    for atom, d in itertools.product(range(3), range(3)):
        mp_, mm_ = _displaced(mol, atom, d, h), _displaced(mol, atom, d, -h)
        for name, g, f in (("J", gJ, lambda m: orc.grad_J(m, D, c)[1]), ("PQ", gQ, lambda m: orc.grad_PQ(m, c, dq)[1])):
            fd = (f(mp_)[0] - f(mm_)[0]) / (2 * h)
            assert abs(g[0, atom, d] - fd) < 2e-7 * np.abs(g[0]).max(), (name, atom, d, g[0, atom, d], fd)


def test_s_functions_of_the_jfit_set_reproduce_the_default_set():
    """A J-fit set that lists exactly one s shell per atom with the default exponents is the default set."""
    mol = _mol_sp()
    m0 = copy.copy(mol)
    m0.jfit = None
    m1 = copy.copy(mol)
    m1.jfit = (np.arange(3), np.zeros(3, dtype=int), mol.aux_exponents.copy())
    rng = np.random.default_rng(2)
    D = rng.standard_normal((2, mol.nao, mol.nao))
    c = rng.standard_normal((2, 3))
    np.testing.assert_array_equal(orc.grad_J(m0, D, c)[0], orc.grad_J(m1, D, c)[0])
    np.testing.assert_allclose(orc.grad_PQ(m0, c, c)[0], orc.grad_PQ(m1, c, c)[0], rtol=0, atol=1e-14)
    np.testing.assert_allclose(orc.metric_J(m1), orc.metric(m0), rtol=1e-14)
    # the K-type calls never see the J-fit set
    Co, Cv, B = rng.standard_normal((mol.nao, 2)), rng.standard_normal((mol.nao, 3)), rng.standard_normal((1, 3, 2, 3))
    np.testing.assert_array_equal(orc.grad_K(mol, Co, Cv, B)[0], orc.grad_K(m0, Co, Cv, B)[0])


def test_fitted_energy_through_the_solve_with_p_functions():
    """The composed RI-J gradient G_J(D, c) - 1/2 G_PQ(c, c), c = M_J^-1 v (Eq. 27) against central differences
    of 1/2 v^T M_J^-1 v with the fit re-solved at every displaced geometry: pins metric_J, vec_J and both gradients with p
    functions against each other through a route none of them shares."""
    mol = _mol_sp()
    rng = np.random.default_rng(21)
    D = rng.standard_normal((1, mol.nao, mol.nao))
    g = orc.grad_RIJ(mol, D)
    M = orc.metric_J(mol)
    assert np.allclose(M, M.T, atol=1e-14) and np.linalg.eigvalsh(M).min() > 0
    h = 5e-6
    for atom, d in itertools.product(range(3), range(3)):
        ep = orc.fit_J(_displaced(mol, atom, d, h), D)[2][0]
        em = orc.fit_J(_displaced(mol, atom, d, -h), D)[2][0]
        fd = (ep - em) / (2 * h)
        assert abs(g[0, atom, d] - fd) < 5e-7 * np.abs(g[0]).max(), (atom, d, g[0, atom, d], fd)
