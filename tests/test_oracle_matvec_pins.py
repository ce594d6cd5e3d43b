"""Pins of the oracle's ris coupling-matrix products (oracle.ris_oracle.coupling_ris / matvec_ris; SURVEY.md 8(f) NEXT-3 and
NEXT-4c; Eqs. 2-5, 20-22) against what the paper and the mathematics fix:
  * the bilinear form of Eq. 39 for products of MO coefficient vectors: X1.K.X2 equals the already pinned
    ris_pair_scalar for the two index orders that give the A-type and the B-type exchange;
  * the Coulomb part with an s + p J-fit set equals twice the pinned fitted energy E_RIJ of D = C_occ X C_vir^T;
  * pure-Python loops over every index on the tiniest case (an index transposed in an einsum string fails here);
  * symmetry of each part, positive semi-definiteness of the Coulomb part, covariance under rotations of the occupied and
    of the virtual orbitals among themselves."""
import numpy as np
import pytest

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import synth


def _mol(seed=5, jfit=True):
    mol = synth.tiny_molecule(seed, [[0, 1], [2, 0], [1]], [[0, 0, 0], [1.8, 0.3, -0.4], [-0.7, 1.6, 0.9]], nprim=2)
    return synth.with_jfit(mol, seed) if jfit else mol


def _orbitals(mol, nocc, nvir, seed):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.standard_normal((mol.nao, nocc + nvir)))
    return np.ascontiguousarray(Q[:, :nocc]), np.ascontiguousarray(Q[:, nocc:])


def test_bilinear_form_equals_the_pinned_pair_scalar_for_both_exchange_orders():
    mol = _mol(jfit=False)
    Co, Cv = _orbitals(mol, 3, 4, 1)
    rng = np.random.default_rng(2)
    X1, X2 = rng.standard_normal((3, 4)), rng.standard_normal((3, 4))
    c_x = 0.37
    D1 = Co @ X1 @ Cv.T
    # D2_rs = C_rj X_jb C_sb: g_{pq,rs} = (pq|rs) - c_x (ps|rq) gives (ia|jb) - c_x (ib|ja): the B-type exchange
    sB = orc.ris_pair_scalar(mol, D1, Co @ X2 @ Cv.T, c_x)
    KB = orc.coupling_ris(mol, Co, Cv, 1.0, 0.0, c_x)
    assert abs(np.einsum("ia,iajb,jb->", X1, KB, X2) - sB) <= 1e-12 * max(1.0, abs(sB))
    # D2_rs = C_rb X_jb C_sj: (ia|bj) - c_x (ij|ba): the A-type exchange
    sA = orc.ris_pair_scalar(mol, D1, Cv @ X2.T @ Co.T, c_x)
    KA = orc.coupling_ris(mol, Co, Cv, 1.0, c_x, 0.0)
    assert abs(np.einsum("ia,iajb,jb->", X1, KA, X2) - sA) <= 1e-12 * max(1.0, abs(sA))
    assert abs(sA - sB) > 1e-3 * abs(sA)          # the two orders are different numbers: the pins are not degenerate


def test_coulomb_part_with_sp_jfit_set_is_twice_the_fitted_energy():
    mol = _mol(jfit=True)
    Co, Cv = _orbitals(mol, 3, 4, 3)
    X = np.random.default_rng(4).standard_normal((3, 4))
    KJ = orc.coupling_ris(mol, Co, Cv, 1.0, 0.0, 0.0)
    D = Co @ X @ Cv.T
    _, _, e = orc.fit_J(mol, D[None])
    got = np.einsum("ia,iajb,jb->", X, KJ, X)
    assert abs(got - 2.0 * e[0]) <= 1e-12 * abs(got)
    # and it differs from the s-only set (the p functions contribute)
    m0 = _mol(jfit=False)
    assert abs(np.einsum("ia,iajb,jb->", X, orc.coupling_ris(m0, Co, Cv, 1.0, 0.0, 0.0), X) - got) > 1e-6 * abs(got)


def test_against_loops_over_every_index():
    mol = synth.with_jfit(synth.tiny_molecule(9, [[0, 1], [0]], [[0, 0, 0], [1.5, 0.5, -0.2]], nprim=2), 9, p_on={0})
    Co, Cv = _orbitals(mol, 2, 2, 5)
    nK, MJ, MK = 2, orc.metric_J(mol), orc.metric(mol)
    nJ = MJ.shape[0]
    IJ = [orc.int3c_J(mol, f) for f in range(nJ)]
    IK = [orc.int3c(mol, P) for P in range(nK)]
    MJi, MKi = np.linalg.inv(MJ), np.linalg.inv(MK)
    nao = mol.nao

    def mo(I, Cl, l, Cr, r):
        return sum(Cl[m, l] * I[m, n] * Cr[n, r] for m in range(nao) for n in range(nao))

    cJ, cKA, cKB = 1.3, 0.4, 0.7
    K = orc.coupling_ris(mol, Co, Cv, cJ, cKA, cKB)
    for i in range(2):
        for a in range(2):
            for j in range(2):
                for b in range(2):
                    ref = 0.0
                    for A in range(nJ):
                        for B in range(nJ):
                            ref += cJ * mo(IJ[A], Co, i, Cv, a) * MJi[A, B] * mo(IJ[B], Co, j, Cv, b)
                    for A in range(nK):
                        for B in range(nK):
                            ref -= cKA * mo(IK[A], Co, i, Co, j) * MKi[A, B] * mo(IK[B], Cv, a, Cv, b)
                            ref -= cKB * mo(IK[A], Co, i, Cv, b) * MKi[A, B] * mo(IK[B], Co, j, Cv, a)
                    assert abs(K[i, a, j, b] - ref) <= 1e-12 * max(1.0, abs(ref)), (i, a, j, b)


def test_symmetry_definiteness_and_orbital_rotations():
    mol = _mol()
    no, nv = 3, 4
    Co, Cv = _orbitals(mol, no, nv, 7)
    rng = np.random.default_rng(8)
    for coef in [(1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0)]:
        K = orc.coupling_ris(mol, Co, Cv, *coef).reshape(no * nv, no * nv)
        assert np.abs(K - K.T).max() <= 1e-13 * np.abs(K).max()
    KJ = orc.coupling_ris(mol, Co, Cv, 1.0, 0.0, 0.0).reshape(no * nv, no * nv)
    assert np.linalg.eigvalsh(0.5 * (KJ + KJ.T)).min() >= -1e-12 * np.abs(KJ).max()
    # sigma(C_occ U, C_vir V; U^T X V) = U^T sigma(C_occ, C_vir; X) V
    U, _ = np.linalg.qr(rng.standard_normal((no, no)))
    V, _ = np.linalg.qr(rng.standard_normal((nv, nv)))
    X = rng.standard_normal((2, no, nv))
    s0 = orc.matvec_ris(mol, Co, Cv, X, 1.1, 0.3, 0.6)
    s1 = orc.matvec_ris(mol, Co @ U, Cv @ V, np.einsum("ij,vjb,bc->vic", U.T, X, V), 1.1, 0.3, 0.6)
    np.testing.assert_allclose(s1, np.einsum("ij,vjb,bc->vic", U.T, s0, V), rtol=0, atol=1e-12 * np.abs(s0).max())
    # linear in X, one vector at a time
    np.testing.assert_allclose(orc.matvec_ris(mol, Co, Cv, X[:1], 1.1, 0.3, 0.6), s0[:1], rtol=0, atol=1e-14 * np.abs(s0).max())
