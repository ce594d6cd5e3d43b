"""Parity of the J-type calls with a J-fit auxiliary set of s AND p functions --
ris_set_jfit, then ris_grad_J, ris_grad_PQ, ris_fit_J, ris_metric_J and the composed RI-J gradient -- against the oracle
(oracle.ris_oracle with mol.jfit), through the C ABI.  Tolerances as in test_gpu_parity.py / test_gpu_fit.py."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import ris_setup, synth

from test_gpu_parity import assert_parity, dev

pytestmark = pytest.mark.gpu
EPS = 2.220446049250313e-16


def _check(mol, D, what, *, fit=True, seed=0):
    rng = np.random.default_rng(1000 + seed)
    nb, n = D.shape[0], synth.naux_jfit(mol)
    c, d = rng.standard_normal((nb, n)), rng.standard_normal((nb, n))
    ctx = ris_setup(mol)
    assert ctx.naux_J == n and ctx.naux == mol.natoms
    gJ = ctx.grad_J(dev(D), dev(c)).cpu().numpy()
    gJ_ref, _ = orc.grad_J(mol, D, c)
    assert_parity(gJ, gJ_ref, what + " J", literal=True)
    gQ = ctx.grad_PQ(dev(c), dev(d)).cpu().numpy()
    gQ_ref, _ = orc.grad_PQ(mol, c, d)
    assert_parity(gQ, gQ_ref, what + " PQ", literal=True)
    M = ctx.metric_J().cpu().numpy()
    M_ref = orc.metric_J(mol)
    np.testing.assert_allclose(M, M_ref, rtol=1e-13, atol=1e-15 * np.abs(M_ref).max())
    # the K-type calls keep the default s set
    np.testing.assert_allclose(ctx.metric().cpu().numpy(), orc.metric(mol), rtol=1e-13, atol=0)
    if fit:
        v, cf = ctx.fit_J(dev(D))
        v, cf = v.cpu().numpy(), cf.cpu().numpy()
        v_ref, c_ref, e_ref = orc.fit_J(mol, D)
        assert_parity(v, v_ref, what + " v")
        cond = np.linalg.cond(M_ref)
        ctol = 64.0 * cond * EPS
        assert np.abs(cf - c_ref).max() <= ctol * np.abs(c_ref).max(), (what, np.abs(cf - c_ref).max(), ctol, cond)
        res = cf @ M_ref - v_ref
        assert np.abs(res).max() <= 1e-12 * np.abs(v_ref).max() * max(1.0, np.abs(M_ref).max()), (what, np.abs(res).max())
        cd = dev(cf)
        g = (ctx.grad_J(dev(D), cd) - 0.5 * ctx.grad_PQ(cd, cd)).cpu().numpy()
        g_ref = orc.grad_RIJ(mol, D)
        assert np.abs(g - g_ref).max() <= max(ctol, 5e-14) * max(1.0, np.abs(orc.grad_J(mol, D, c_ref)[0]).max()), what
    ctx.close()


@pytest.mark.parametrize("cfg", [1, 2])
def test_jfit_sp_small_configs(cfg):
    wl = synth.make_workload(cfg)
    _check(synth.with_jfit(wl.mol, cfg), wl.D, f"config {cfg} s+p", seed=cfg)


def test_jfit_sp_all_classes_up_to_f_and_many_states():
    mol = synth.tiny_molecule(21, [[0, 1, 2, 3], [3, 2, 0], [1, 3], [0]],
                              [[0, 0, 0], [1.9, 0.4, -0.3], [-0.8, 1.7, 1.0], [0.5, -2.2, 1.4]], nprim=2)
    rng = np.random.default_rng(9)
    _check(synth.with_jfit(mol, 5), rng.standard_normal((7, mol.nao, mol.nao)), "all classes s+p")


def test_jfit_ragged_sets_and_reset():
    """p shells on some atoms only (ragged lists: 2 p functions per component, 5 s), an atom without any function, a set of
    p functions only; a second ris_set_jfit on the same context replaces the first."""
    mol = synth.tiny_molecule(8, [[0, 1], [2], [1, 1], [0], [2, 0]],
                              [[0, 0, 0], [2.1, 0.2, -0.4], [-1.0, 1.9, 0.8], [0.7, -2.0, 1.5], [3.0, 2.0, 1.0]])
    rng = np.random.default_rng(3)
    D = rng.standard_normal((2, mol.nao, mol.nao))
    m1 = synth.with_jfit(mol, 1, p_on={1, 3})
    _check(m1, D, "ragged")
    m2 = synth.with_jfit(mol, 2)
    m2.jfit = (np.array([0, 2, 4], dtype=np.int32), np.array([1, 1, 1], dtype=np.int32), np.array([0.3, 0.5, 0.9]))
    _check(m2, D, "p only, atoms 1 and 3 bare")
    ctx = ris_setup(m1)
    c = rng.standard_normal((2, synth.naux_jfit(m2)))
    ctx.set_jfit(*m2.jfit)
    assert ctx.naux_J == 9
    assert_parity(ctx.grad_J(dev(D), dev(c)).cpu().numpy(), orc.grad_J(m2, D, c)[0], "reset J", literal=True)
    ctx.close()


def test_jfit_s_only_set_equals_default_set():
    wl = synth.make_workload(2)
    mol = wl.mol
    m1 = synth.with_jfit(mol, 0, p_on=set())
    c0, c1 = ris_setup(mol), ris_setup(m1)
    D, c = dev(wl.D), dev(wl.c_aux)
    g0, g1 = c0.grad_J(D, c).cpu().numpy(), c1.grad_J(D, c).cpu().numpy()
    assert np.abs(g0 - g1).max() <= 5e-15 * np.abs(g0).max()
    q0, q1 = c0.grad_PQ(c, dev(wl.d_aux)).cpu().numpy(), c1.grad_PQ(c, dev(wl.d_aux)).cpu().numpy()
    assert np.abs(q0 - q1).max() <= 5e-15 * np.abs(q0).max()
    c0.close(); c1.close()


def test_jfit_sp_full_size_config3():
    """Config 3 (100 atoms, 1100 AO, 5 states; 400 J-fit functions) at full size: J on sampled atoms, PQ in full, v on sampled
    functions of every type."""
    wl = synth.make_workload(3)
    mol = synth.with_jfit(wl.mol, 3)
    n = synth.naux_jfit(mol)
    rng = np.random.default_rng(33)
    nb = wl.D.shape[0]
    c, d = rng.standard_normal((nb, n)), rng.standard_normal((nb, n))
    ctx = ris_setup(mol, schwarz_tol=wl.schwarz_tol)
    gJ = ctx.grad_J(dev(wl.D), dev(c)).cpu().numpy()
    atoms = [0, 13, 50, 99]
    ref, _ = orc.grad_J(mol, wl.D, c, atoms=atoms)
    assert np.isnan(ref).sum() == 3 * nb * (mol.natoms - len(atoms))        # unsampled rows are NaN: skipped by assert_parity
    assert_parity(gJ, ref, "config 3 s+p J (sampled atoms)", literal=True)
    assert np.abs(gJ.sum(axis=1)).max() <= 1e-11 * np.abs(gJ).max()
    gQ = ctx.grad_PQ(dev(c), dev(d)).cpu().numpy()
    assert_parity(gQ, orc.grad_PQ(mol, c, d)[0], "config 3 s+p PQ", literal=True)
    v, cf = ctx.fit_J(dev(wl.D))
    v, cf = v.cpu().numpy(), cf.cpu().numpy()
    import ctypes as C
    h = orc._Held(mol, jfit=True)
    D = np.ascontiguousarray(wl.D, dtype=np.float64)
    one = np.ones(nb)
    scale = np.abs(v).max()
    for P in (0, 1, 2, 3, 201, 202, 399):
        g = np.zeros((nb, h.natoms, 3), dtype=np.longdouble)
        e = np.zeros(nb, dtype=np.longdouble)
        assert orc.lib().ris_oracle_contract_P(C.byref(h.c), P, nb, D.ctypes.data, one.ctypes.data, None, 0.0,
                                               g.ctypes.data, e.ctypes.data) == 0
        r = e.astype(np.float64)
        assert np.all(np.abs(v[:, P] - r) <= 1e-10 * np.abs(r) + 1e-12 * scale), (P, v[:, P], r)
    M_ref = orc.metric_J(mol)
    res = cf @ M_ref - v
    assert np.abs(res).max() <= 1e-11 * np.abs(v).max() * max(1.0, np.abs(M_ref).max())
    ctx.close()
