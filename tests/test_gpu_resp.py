"""Parity of the coupling-matrix products (ris_resp_setup / ris_resp_matvec; SURVEY.md 8(f) NEXT-3, NEXT-4c; Eqs. 2-5, 20-22,
PAPER.md:36-53, 115-123, 213-217) with the oracle's dense definition (oracle.ris_oracle.matvec_ris), through the C ABI.

Tolerance: sigma is a sum of products of fitted tensors, M^-1 enters once per term; two backward-stable solvers differ by
~cond(M) eps, so sigma is compared at 64 max(cond(M_J), cond(M_K)) eps of its scale (reading R-cond), never
looser than 5e-14 of the scale; the Coulomb-only and exchange-only products are checked separately so that a small term
cannot hide behind a large one."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import RisError, ris_setup, synth

from test_gpu_parity import dev

pytestmark = pytest.mark.gpu
EPS = 2.220446049250313e-16
COEFS = [(1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0), (2.0, 0.25, 0.25), (0.0, 0.2, -0.2)]


def _orbitals(mol, nocc, nvir, seed):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.standard_normal((mol.nao, nocc + nvir)))
    return np.ascontiguousarray(Q[:, :nocc]), np.ascontiguousarray(Q[:, nocc:])


def _check(mol, nocc, nvir, nvec, what, seed=0, coefs=COEFS):
    Co, Cv = _orbitals(mol, nocc, nvir, seed)
    X = np.random.default_rng(seed + 1).standard_normal((nvec, nocc, nvir))
    ctx = ris_setup(mol)
    ctx.resp_setup(dev(Co), dev(Cv))
    tol = max(5e-14, 64.0 * EPS * max(np.linalg.cond(orc.metric_J(mol)), np.linalg.cond(orc.metric(mol))))
    for cJ, cKA, cKB in coefs:
        got = ctx.resp_matvec(dev(X), cJ, cKA, cKB).cpu().numpy()
        ref = orc.matvec_ris(mol, Co, Cv, X, cJ, cKA, cKB)
        err = np.abs(got - ref).max() / np.abs(ref).max()
        assert err <= tol, (what, (cJ, cKA, cKB), err, tol)
    ctx.close()


def test_matvec_config1_sp_jfit():
    wl = synth.make_workload(1)
    _check(synth.with_jfit(wl.mol, 1), 5, 20, 3, "config 1 s+p")


def test_matvec_all_classes_odd_dimensions_many_vectors():
    """f shells, odd nocc / nvir (padded rows), 11 vectors (two passes of the Coulomb kernels), default and s+p sets."""
    mol = synth.tiny_molecule(21, [[0, 1, 2, 3], [3, 2, 0], [1, 3], [0]],
                              [[0, 0, 0], [1.9, 0.4, -0.3], [-0.8, 1.7, 1.0], [0.5, -2.2, 1.4]], nprim=2)
    _check(mol, 7, 13, 11, "all classes, default set", seed=3)
    _check(synth.with_jfit(mol, 2, p_on={0, 2}), 5, 9, 2, "all classes, ragged s+p", seed=4)


def test_matvec_config2_sampled_elements():
    """Config 2 (30 atoms, 300 AO, nocc 42, nvir 84, s+p J-fit set of 120 functions): the dense oracle matrix would be
    (42*84)^2 doubles; the oracle's definition is evaluated for sampled sigma elements instead."""
    wl = synth.make_workload(2)
    mol = synth.with_jfit(wl.mol, 2)
    Co, Cv = np.ascontiguousarray(wl.C_occ), np.ascontiguousarray(wl.C_vir)
    nocc, nvir = Co.shape[1], Cv.shape[1]
    X = np.random.default_rng(5).standard_normal((2, nocc, nvir))
    ctx = ris_setup(mol)
    ctx.resp_setup(dev(Co), dev(Cv))
    nK, MJ, MK = mol.natoms, orc.metric_J(mol), orc.metric(mol)
    IK = np.stack([orc.int3c(mol, P) for P in range(nK)])
    IJ = np.stack([orc.int3c_J(mol, f) for f in range(MJ.shape[0])])
    TJ = orc.mo_tensor(IJ, Co, Cv)
    Too, Tov, Tvv = orc.mo_tensor(IK, Co, Co), orc.mo_tensor(IK, Co, Cv), orc.mo_tensor(IK, Cv, Cv)
    MJi, MKi = np.linalg.inv(MJ), np.linalg.inv(MK)
    tol = max(5e-14, 64.0 * EPS * max(np.linalg.cond(MJ), np.linalg.cond(MK)))
    samples = [(0, 0), (41, 83), (17, 5), (3, 60), (40, 1)]
    for cJ, cKA, cKB in [(1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0), (2.0, 0.25, 0.25)]:
        got = ctx.resp_matvec(dev(X), cJ, cKA, cKB).cpu().numpy()
        scale = np.abs(got).max()
        for i, a in samples:
            # row (i, a) of the matrix of coupling_ris, written out
            row = cJ * np.einsum("A,AB,Bjb->jb", TJ[:, i, a], MJi, TJ)
            row -= cKA * np.einsum("Aj,AB,Bb->jb", Too[:, i, :], MKi, Tvv[:, a, :])
            row -= cKB * np.einsum("Ab,AB,Bj->jb", Tov[:, i, :], MKi, Tov[:, :, a])
            ref = np.einsum("jb,vjb->v", row, X)
            assert np.abs(got[:, i, a] - ref).max() <= tol * scale, ((cJ, cKA, cKB), (i, a), got[:, i, a], ref)
    # symmetric matrix: X1 . sigma(X2) = X2 . sigma(X1)
    s = ctx.resp_matvec(dev(X), 2.0, 0.25, 0.25).cpu().numpy()
    assert abs(np.sum(X[0] * s[1]) - np.sum(X[1] * s[0])) <= 1e-11 * abs(np.sum(X[0] * s[1]))
    ctx.close()


def test_matvec_errors_and_reuse():
    wl = synth.make_workload(1)
    ctx = ris_setup(wl.mol)
    X = dev(np.ones((1, 5, 20)))
    with pytest.raises(RisError):
        ctx.resp_matvec(X, 1.0, 0.0, 0.0)
    Co, Cv = _orbitals(wl.mol, 5, 20, 0)
    ctx.resp_setup(dev(Co), dev(Cv))
    a = ctx.resp_matvec(X, 1.0, 0.5, 0.5).cpu().numpy()
    ctx.resp_setup(dev(Co), dev(Cv))                      # rebuild on the same context
    b = ctx.resp_matvec(X, 1.0, 0.5, 0.5).cpu().numpy()
    assert np.array_equal(a, b)                           # deterministic
    z = ctx.resp_matvec(X, 0.0, 0.0, 0.0).cpu().numpy()
    assert np.all(z == 0.0)
    ctx.close()
