"""Pins of the oracle's spherical-harmonic shells (NEXT-4b; "def2-TZVP", a spherical basis; SURVEY.md 8(f)
NEXT-4; reading R-sph).  None of them retypes the closed formula the oracle builds its table from:

  * values of sqrt(4 pi/(2l+1)) r^l Y_lm (scipy's complex spherical harmonics, combined into the real ones) at random points;
  * every S_lm is a harmonic polynomial (Laplacian computed on the monomial coefficients);
  * orthogonality and the common norm of the 2l+1 functions of a shell under a Gaussian weight (closed-form monomial
    moments), 4 pi/(2l+1) int r^{2l+2} exp(-2 a r^2) dr;
  * one three-centre integral over a spherical d / f function pair against brute-force 3-D Gauss-Hermite quadrature with
    the function values taken from scipy;
  * rotation of the whole problem: the gradient in the spherical basis with a rotation-invariant density (identity blocks)
    rotates like a vector.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import synth


def _comps(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def _real_sph(l, m, xyz):
    """sqrt(4 pi/(2l+1)) r^l Y_lm^{real}(r) from scipy's complex Y_l^m (Condon-Shortley phase)."""
    from scipy.special import sph_harm_y
    x, y, z = xyz[..., 0], xyz[..., 1], xyz[..., 2]
    r = np.sqrt(x * x + y * y + z * z)
    theta, phi = np.arccos(z / r), np.arctan2(y, x)
    am = abs(m)
    Y = sph_harm_y(l, am, theta, phi)
    if m == 0:
        real = Y.real
    elif m > 0:
        real = math.sqrt(2.0) * (-1) ** m * Y.real
    else:
        real = math.sqrt(2.0) * (-1) ** m * Y.imag
    return math.sqrt(4 * math.pi / (2 * l + 1)) * r ** l * real


@pytest.mark.parametrize("l", [0, 1, 2, 3])
def test_table_against_scipy_spherical_harmonics(l):
    rng = np.random.default_rng(10 + l)
    pts = rng.normal(size=(40, 3))
    T = orc.solid_harmonic_cart(l)
    mono = np.stack([pts[:, 0] ** cx * pts[:, 1] ** cy * pts[:, 2] ** cz for cx, cy, cz in _comps(l)], -1)
    for m in range(-l, l + 1):
        got = mono @ T[m + l]
        ref = _real_sph(l, m, pts)
        assert np.abs(got - ref).max() <= 1e-13 * max(1.0, np.abs(ref).max()), (l, m)


def test_low_orders_are_the_textbook_polynomials():
    T1 = orc.solid_harmonic_cart(1)          # order m = -1, 0, 1 -> y, z, x
    assert np.array_equal(T1, np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]], dtype=float))
    T2 = orc.solid_harmonic_cart(2)          # cart order xx xy xz yy yz zz
    assert np.allclose(T2[2], [-0.5, 0, 0, -0.5, 0, 1.0], atol=1e-15)            # z^2 - (x^2 + y^2)/2
    assert np.allclose(T2[4], [math.sqrt(3) / 2, 0, 0, -math.sqrt(3) / 2, 0, 0], atol=1e-15)
    assert np.allclose(T2[0], [0, math.sqrt(3), 0, 0, 0, 0], atol=1e-15)


@pytest.mark.parametrize("l", [2, 3])
def test_harmonic_polynomials(l):
    comps = _comps(l)
    low = _comps(l - 2)
    T = orc.solid_harmonic_cart(l)
    for m in range(2 * l + 1):
        lap = np.zeros(len(low))
        for coef, c in zip(T[m], comps):
            for d in range(3):
                if c[d] >= 2:
                    e = list(c); e[d] -= 2
                    lap[low.index(tuple(e))] += coef * c[d] * (c[d] - 1)
        assert np.abs(lap).max() <= 1e-14, (l, m, lap)


def _dfact(n):
    return 1.0 if n <= 0 else n * _dfact(n - 2)


def _moment(n, g):
    """int x^n exp(-g x^2) dx"""
    return 0.0 if n % 2 else _dfact(n - 1) / (2 * g) ** (n // 2) * math.sqrt(math.pi / g)


@pytest.mark.parametrize("l", [1, 2, 3])
def test_orthogonal_with_a_common_norm_under_a_gaussian_weight(l):
    a = 0.7
    comps = _comps(l)
    G = np.array([[math.prod(_moment(c1[d] + c2[d], 2 * a) for d in range(3)) for c2 in comps] for c1 in comps])
    T = orc.solid_harmonic_cart(l)
    S = T @ G @ T.T
    # 4 pi/(2l+1) int_0^inf r^{2l+2} exp(-2 a r^2) dr,  int r^{2n} e^{-g r^2} = (2n-1)!!/(2 (2g)^n) sqrt(pi/g)
    n = l + 1
    norm = 4 * math.pi / (2 * l + 1) * _dfact(2 * n - 1) / (2 * (4 * a) ** n) * math.sqrt(math.pi / (2 * a))
    assert np.abs(S - norm * np.eye(2 * l + 1)).max() <= 1e-14 * norm


def test_sph_matrix_blocks_and_sizes():
    mol = synth.tiny_molecule(3, [[0, 2], [3, 1]], np.array([[0.0, 0.0, 0.0], [1.5, 0.3, -0.2]]))
    U = orc.sph_matrix(mol)
    assert U.shape == (1 + 5 + 7 + 3, 1 + 6 + 10 + 3) == (orc.nao_sph(mol), mol.nao)
    assert np.array_equal(U[0:1, 0:1], [[1.0]])
    assert np.array_equal(U[1:6, 1:7], orc.solid_harmonic_cart(2))
    assert np.array_equal(U[6:13, 7:17], orc.solid_harmonic_cart(3))
    assert np.count_nonzero(U[1:6, 7:]) == 0 and np.count_nonzero(U[6:13, :7]) == 0


def _quad3c_sph(la, ma, lb, mb, a, b, alpha, A, B, Cc, n=48):
    """int S_{la ma}(r-A) e^{-a|r-A|^2} S_{lb mb}(r-B) e^{-b|r-B|^2} V_C(r) dr by 3-D Gauss-Hermite quadrature on the product
    Gaussian; V_C(r) = (pi/alpha)^{3/2} erf(sqrt(alpha)|r-C|)/|r-C|; angular factors from scipy."""
    from scipy.special import erf
    p = a + b
    P = (a * A + b * B) / p
    Kab = math.exp(-a * b / p * np.dot(A - B, A - B))
    x, w = np.polynomial.hermite.hermgauss(n)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    W = w[:, None, None] * w[None, :, None] * w[None, None, :]
    r = np.stack([X, Y, Z], -1) / math.sqrt(p) + P
    ang = _real_sph(la, ma, r - A) * _real_sph(lb, mb, r - B)
    dist = np.linalg.norm(r - Cc, axis=-1)
    V = (math.pi / alpha) ** 1.5 * erf(math.sqrt(alpha) * dist) / dist
    return Kab * p ** -1.5 * np.sum(W * ang * V)


@pytest.mark.parametrize("la,lb", [(2, 1), (3, 2)])
def test_spherical_three_centre_integral_against_quadrature(la, lb):
    """(mu nu|P) of a one-primitive molecule over spherical functions vs the quadrature, a few (m, m') pairs."""
    a, b, alpha = 0.9, 0.6, 0.35
    A, B = np.array([0.2, -0.1, 0.3]), np.array([-0.4, 0.5, 0.1])
    mol = synth.Molecule(coords=np.stack([A, B]), Z=np.array([6, 6], dtype=np.int32), shell_atom=np.array([0, 1], dtype=np.int32),
                         shell_l=np.array([la, lb], dtype=np.int32), shell_nprim=np.array([1, 1], dtype=np.int32),
                         shell_prim_off=np.array([0, 1], dtype=np.int32), prim_exp=np.array([a, b]), prim_coef=np.array([1.0, 1.0]),
                         aux_exponents=np.array([alpha, 0.5]))
    I = orc.int3c_sph(mol, 0)                  # aux function 0 sits on atom 0 (centre A); N_P (2 alpha/pi)^{3/4} included
    NP = (2 * alpha / math.pi) ** 0.75
    na = 2 * la + 1
    for ma, mb in [(-la, -lb), (0, 0), (la, lb - 1), (1, -1), (-2 if la >= 2 else 0, lb)]:
        got = I[ma + la, na + mb + lb]
        ref = NP * _quad3c_sph(la, ma, lb, mb, a, b, alpha, A, B, A)
        assert abs(got - ref) <= 5e-11 * max(1.0, abs(ref)), (ma, mb, got, ref)


def test_gradient_rotates_like_a_vector_for_an_invariant_density():
    """A density that is a multiple of the identity inside every (shell, shell') block of equal l is invariant under
    rotations in the spherical basis (the 2l+1 functions carry an orthogonal representation, their common norm pinned above),
    so rotating the geometry must rotate the J gradient: g(R x) = R g(x).  In the Cartesian d / f basis the same block
    pattern is NOT invariant -- the test would fail with U left out."""
    rng = np.random.default_rng(5)
    coords = np.array([[0.0, 0.0, 0.0], [1.8, 0.4, -0.3], [-0.7, 1.6, 0.9]])
    ls = [[0, 2], [1, 3], [2, 3]]
    mol = synth.tiny_molecule(11, ls, coords)
    n = orc.nao_sph(mol)
    off = np.concatenate([[0], np.cumsum([2 * int(l) + 1 for l in mol.shell_l])])
    D = np.zeros((n, n))
    for i, li in enumerate(mol.shell_l):
        for j, lj in enumerate(mol.shell_l):
            if li == lj:
                D[off[i]:off[i + 1], off[j]:off[j + 1]] = rng.normal() * np.eye(2 * int(li) + 1)
    c = rng.normal(size=(1, mol.natoms))
    g0 = orc.grad_J_sph(mol, D[None], c)[0][0]
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    mol_r = synth.tiny_molecule(11, ls, coords @ Q.T)
    g1 = orc.grad_J_sph(mol_r, D[None], c)[0][0]
    scale = np.abs(g0).max()
    assert np.abs(g1 - g0 @ Q.T).max() <= 1e-11 * scale
    # the Cartesian basis with the same block pattern is not rotation invariant (d and f shells present)
    Dc = np.zeros((mol.nao, mol.nao))
    offc = np.concatenate([[0], np.cumsum([synth.ncart(int(l)) for l in mol.shell_l])])
    for i, li in enumerate(mol.shell_l):
        for j, lj in enumerate(mol.shell_l):
            if li == lj:
                Dc[offc[i]:offc[i + 1], offc[j]:offc[j + 1]] = np.eye(synth.ncart(int(li)))
    h0 = orc.grad_J(mol, Dc[None], c)[0][0]
    h1 = orc.grad_J(mol_r, Dc[None], c)[0][0]
    assert np.abs(h1 - h0 @ Q.T).max() > 1e-6 * np.abs(h0).max()
