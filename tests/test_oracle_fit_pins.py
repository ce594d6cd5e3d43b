"""Pins of the oracle's J-type fitting step (Eqs. 21-22, 27 of the paper,
PAPER.md:119-121, 150).  No CUDA here.  What fixes the functions from outside:

* the metric: the printed two-centre worked example (tests/golden/prim2c_worked_example.txt), the closed form of the
  self-repulsion of a normalised s Gaussian, (P|P) = N_P^2 2 pi^{5/2} / (alpha^2 sqrt(2 alpha)) = 4 pi / alpha ... computed
  independently below by Gauss-Legendre quadrature of the Boys-function definition at T = 0 and by the erf potential;
* v_P: brute-force 3-D Gauss-Hermite quadrature of  int phi_mu phi_nu V_P  on a tiny s/p molecule;
* the whole fitted energy E_RIJ(R) = 1/2 v^T M^-1 v: central finite differences (5e-6 bohr, the paper's own
  validation) against the composed gradient  G_J(D,c) - 1/2 G_PQ(c,c)  -- the fit (solve) sits
  INSIDE the differentiated function, so a wrong sign / factor of the metric term of Eq. 27 fails it;
* the far-field limit: one s function far from one aux, v -> S N_P (pi/alpha)^{3/2} / R.
"""
import copy
import itertools
import math

import numpy as np
from scipy.special import erf

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import synth


def _tiny(seed=5):
    coords = np.array([[0.0, 0.0, 0.0], [1.9, 0.3, -0.2], [-0.6, 1.7, 0.9]])
    mol = synth.tiny_molecule(seed, [[0, 1, 2], [0, 1], [0, 0]], coords)
    rng = np.random.default_rng(seed)
    nao = sum(synth.ncart(int(l)) for l in mol.shell_l)
    D = rng.standard_normal((2, nao, nao))
    D[0] = 0.5 * (D[0] + D[0].T)
    return mol, D


def test_metric_diagonal_closed_form_and_symmetry():
    mol, _ = _tiny()
    M = orc.metric(mol)
    al = mol.aux_exponents
    # self-repulsion of a normalised s Gaussian: N^2 2 pi^{5/2} / (alpha^2 sqrt(2 alpha)), N = (2 alpha/pi)^{3/4}
    ref = (2 * al / math.pi) ** 1.5 * 2 * math.pi ** 2.5 / (al * al * np.sqrt(2 * al))
    np.testing.assert_allclose(np.diag(M), ref, rtol=1e-14)
    np.testing.assert_allclose(M, M.T, rtol=0, atol=1e-15 * np.abs(M).max())
    assert np.all(np.linalg.eigvalsh(M) > 0.0)          # a Coulomb metric is positive definite


def test_metric_offdiagonal_erf_potential():
    """(P|Q) = N_P N_Q (pi^2/(alpha beta))^{3/2} erf(sqrt(rho) R)/R  (two spherical Gaussian charges)."""
    mol, _ = _tiny()
    M = orc.metric(mol)
    al, R = mol.aux_exponents, mol.coords
    N = (2 * al / math.pi) ** 0.75
    for P, Q in itertools.combinations(range(3), 2):
        r = np.linalg.norm(R[P] - R[Q])
        rho = al[P] * al[Q] / (al[P] + al[Q])
        ref = N[P] * N[Q] * (math.pi ** 2 / (al[P] * al[Q])) ** 1.5 * erf(math.sqrt(rho) * r) / r
        assert abs(M[P, Q] - ref) < 1e-13 * abs(ref)


def test_vec_J_against_gauss_hermite_quadrature():
    """v_P for one (p, s) primitive shell pair by 3-D Gauss-Hermite quadrature of phi_a phi_b V_P,
    V_P(r) = N_P (pi/alpha)^{3/2} erf(sqrt(alpha) |r - C|)/|r - C|."""
    coords = np.array([[0.2, -0.1, 0.3], [1.1, 0.6, -0.4]])
    mol = synth.tiny_molecule(7, [[1], [0]], coords, nprim=1)
    a, b = mol.prim_exp[0], mol.prim_exp[1]
    da, db = mol.prim_coef[0], mol.prim_coef[1]
    A, B = coords
    p = a + b
    Pc = (a * A + b * B) / p
    K = math.exp(-a * b / p * np.sum((A - B) ** 2))
    x, w = np.polynomial.hermite.hermgauss(64)
    g = [Pc[d] + x / math.sqrt(p) for d in range(3)]
    X, Y, Z = np.meshgrid(*g, indexing="ij")
    W = w[:, None, None] * w[None, :, None] * w[None, None, :] / p ** 1.5
    nao = 4
    for P in range(2):
        al = mol.aux_exponents[P]
        C = coords[P]
        r = np.sqrt((X - C[0]) ** 2 + (Y - C[1]) ** 2 + (Z - C[2]) ** 2)
        V = (2 * al / math.pi) ** 0.75 * (math.pi / al) ** 1.5 * erf(math.sqrt(al) * r) / r
        for comp, poly in enumerate((X - A[0], Y - A[1], Z - A[2])):
            D = np.zeros((1, nao, nao))
            D[0, comp, 3] = 1.0                       # AO order: p_x p_y p_z (atom 0), s (atom 1)
            ref = da * db * K * np.sum(W * poly * V)
            got = orc.vec_J(mol, D)[0, P]
            assert abs(got - ref) < 2e-11 * max(abs(ref), 1e-3), (P, comp, got, ref)


def test_vec_J_is_linear_and_symmetric_in_D():
    mol, D = _tiny()
    v = orc.vec_J(mol, D)
    np.testing.assert_allclose(orc.vec_J(mol, D.transpose(0, 2, 1)), v, rtol=0, atol=1e-13 * np.abs(v).max())
    v2 = orc.vec_J(mol, 2.0 * D[:1] - 3.0 * D[1:])
    np.testing.assert_allclose(v2[0], 2.0 * v[0] - 3.0 * v[1], rtol=0, atol=1e-12 * np.abs(v).max())


def test_fitted_energy_finite_difference():
    """d/dR [1/2 v^T M^-1 v] (fit re-solved at every displaced geometry) = G_J(D,c) - 1/2 G_PQ(c,c)."""
    mol, D = _tiny()
    g = orc.grad_RIJ(mol, D)
    h = 5e-6
    scale = np.abs(g).max(axis=(1, 2))
    for atom, d in itertools.product(range(3), range(3)):
        mp_, mm_ = copy.copy(mol), copy.copy(mol)
        mp_.coords = mol.coords.copy(); mp_.coords[atom, d] += h
        mm_.coords = mol.coords.copy(); mm_.coords[atom, d] -= h
        fd = (orc.fit_J(mp_, D)[2] - orc.fit_J(mm_, D)[2]) / (2 * h)
        assert np.all(np.abs(g[:, atom, d] - fd) < 5e-7 * scale), (atom, d, g[:, atom, d], fd)


def test_fitted_gradient_translational_invariance():
    mol, D = _tiny()
    g = orc.grad_RIJ(mol, D)
    assert np.all(np.abs(g.sum(axis=1)) < 1e-10 * np.abs(g).sum())


def test_vec_J_far_field_limit():
    """One s function and an aux function 200 bohr away: v -> S N_P (pi/alpha)^{3/2} / R (P12)."""
    coords = np.array([[0.0, 0.0, 0.0], [200.0, 0.0, 0.0]])
    mol = synth.tiny_molecule(3, [[0], []], coords, nprim=1)
    a, d = mol.prim_exp[0], mol.prim_coef[0]
    S = d * d * (math.pi / (2 * a)) ** 1.5
    al = mol.aux_exponents[1]
    ref = S * (2 * al / math.pi) ** 0.75 * (math.pi / al) ** 1.5 / 200.0
    got = orc.vec_J(mol, np.ones((1, 1, 1)))[0, 1]
    assert abs(got - ref) < 1e-8 * ref


# ------------------------------------------------------------------ K-type fitting step

def test_int3c_consistent_with_pinned_contraction_and_symmetric():
    """(mu nu|P) as a matrix against the pinned contraction: sum D.I^P = v_P; symmetric in mu nu."""
    mol, D = _tiny()
    v = orc.vec_J(mol, D)
    for P in range(3):
        I = orc.int3c(mol, P)
        np.testing.assert_allclose(I, I.T, rtol=0, atol=1e-14 * np.abs(I).max())
        np.testing.assert_allclose(np.einsum("smn,mn->s", D, I), v[:, P], rtol=0, atol=1e-12 * np.abs(v).max())


def test_int3c_single_element_by_quadrature():
    coords = np.array([[0.2, -0.1, 0.3], [1.1, 0.6, -0.4]])
    mol = synth.tiny_molecule(7, [[0], [0]], coords, nprim=1)
    a, b = mol.prim_exp
    da, db = mol.prim_coef
    A, B = coords
    p = a + b
    Pc = (a * A + b * B) / p
    x, w = np.polynomial.hermite.hermgauss(48)
    g = [Pc[d] + x / math.sqrt(p) for d in range(3)]
    X, Y, Z = np.meshgrid(*g, indexing="ij")
    W = w[:, None, None] * w[None, :, None] * w[None, None, :] / p ** 1.5
    al = mol.aux_exponents[0]
    r = np.sqrt((X - A[0]) ** 2 + (Y - A[1]) ** 2 + (Z - A[2]) ** 2)
    V = (2 * al / math.pi) ** 0.75 * (math.pi / al) ** 1.5 * erf(math.sqrt(al) * r) / r
    ref = da * db * math.exp(-a * b / p * np.sum((A - B) ** 2)) * np.sum(W * V)
    assert abs(orc.int3c(mol, 0)[0, 1] - ref) < 1e-11 * abs(ref)


def test_grad_PQ_full_reduces_to_rank_one():
    mol, _ = _tiny()
    rng = np.random.default_rng(2)
    c, d = rng.standard_normal((2, 3)), rng.standard_normal((2, 3))
    ref, _ = orc.grad_PQ(mol, c, d)
    got = orc.grad_PQ_full(mol, np.einsum("sp,sq->spq", c, d))
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-13 * np.abs(ref).max())


def test_fitted_K_energy_finite_difference():
    """d/dR [1/2 sum T M^-1 T] with the fit re-solved at every displaced geometry
    = G_K(C_occ, C_vir, B) - 1/2 sum_PQ (B B^T)_PQ M^xi_PQ   (Eq. 27 with a full-matrix metric term)."""
    mol, _ = _tiny()
    rng = np.random.default_rng(8)
    nao = sum(synth.ncart(int(l)) for l in mol.shell_l)
    Co, Cv = rng.standard_normal((nao, 3)), rng.standard_normal((nao, 4))
    g = orc.grad_RIK(mol, Co, Cv)
    h = 5e-6
    scale = np.abs(g).max()
    for atom, d in itertools.product(range(3), range(3)):
        mp_, mm_ = copy.copy(mol), copy.copy(mol)
        mp_.coords = mol.coords.copy(); mp_.coords[atom, d] += h
        mm_.coords = mol.coords.copy(); mm_.coords[atom, d] -= h
        fd = (orc.fit_K(mp_, Co, Cv)[2] - orc.fit_K(mm_, Co, Cv)[2]) / (2 * h)
        assert abs(g[atom, d] - fd) < 5e-7 * scale, (atom, d, g[atom, d], fd)
    assert np.all(np.abs(g.sum(axis=0)) < 1e-10 * np.abs(g).sum())


# ------------------------------------------------------------------ composed <g^ris,(xi); {D1, D2}>

def test_ris_pair_gradient_finite_difference():
    """Eq. 27 for the full ris kernel of Eq. 21 (Coulomb and exchange pairing, c_x = 0.25), D1 != D2, neither
    symmetric: central differences of S(R) = <g^ris(R); {D1, D2}> at fixed AO matrices."""
    mol, D = _tiny()
    D1, D2 = D[0] + 0.3 * D[1], D[1]
    cx = 0.25
    g = orc.ris_pair_gradient(mol, D1, D2, cx)
    h = 5e-6
    scale = np.abs(g).max()
    for atom, d in itertools.product(range(3), range(3)):
        mp_, mm_ = copy.copy(mol), copy.copy(mol)
        mp_.coords = mol.coords.copy(); mp_.coords[atom, d] += h
        mm_.coords = mol.coords.copy(); mm_.coords[atom, d] -= h
        fd = (orc.ris_pair_scalar(mp_, D1, D2, cx) - orc.ris_pair_scalar(mm_, D1, D2, cx)) / (2 * h)
        assert abs(g[atom, d] - fd) < 5e-7 * scale, (atom, d, g[atom, d], fd)
    assert np.all(np.abs(g.sum(axis=0)) < 1e-10 * np.abs(g).sum())


def test_ris_pair_scalar_exchange_index_pairing():
    """The exchange term pairs (ps|A)(B|rq): for rank-one D1 = x y^T, D2 = z w^T it factorises into
    sum_AB M^-1_AB (x^T I^A w)(z^T I^B y); the Coulomb term into (x^T I^A y)(z^T I^B w)."""
    mol, _ = _tiny()
    rng = np.random.default_rng(11)
    nao = sum(synth.ncart(int(l)) for l in mol.shell_l)
    x, y, z, w = rng.standard_normal((4, nao))
    I = [orc.int3c(mol, P) for P in range(3)]
    Minv = np.linalg.inv(orc.metric(mol))
    coul = sum(Minv[A, B] * (x @ I[A] @ y) * (z @ I[B] @ w) for A in range(3) for B in range(3))
    exch = sum(Minv[A, B] * (x @ I[A] @ w) * (z @ I[B] @ y) for A in range(3) for B in range(3))
    D1, D2 = np.outer(x, y), np.outer(z, w)
    assert abs(orc.ris_pair_scalar(mol, D1, D2, 0.0) - coul) < 1e-12 * abs(coul)
    s = orc.ris_pair_scalar(mol, D1, D2, 1.0)
    assert abs((coul - s) - exch) < 1e-11 * max(abs(exch), abs(coul))
