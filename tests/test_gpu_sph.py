"""Spherical-harmonic shells (ris_options.spherical) through the C ABI against the
oracle's spherical definitions (oracle.ris_oracle.grad_J_sph / grad_K_sph / sph_matrix, pinned in
tests/test_oracle_sph_pins.py).  Tolerances: those of test_gpu_parity.py (gradients) and test_gpu_fit.py (fitted quantities)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import RisError, ris_setup, synth

from test_gpu_parity import assert_parity, dev

pytestmark = pytest.mark.gpu
EPS = 2.220446049250313e-16


def _inputs(mol, seed, nb, nocc, nvir):
    rng = np.random.default_rng(seed)
    n, naux = orc.nao_sph(mol), mol.natoms
    return dict(D=rng.standard_normal((nb, n, n)), c=rng.standard_normal((nb, naux)), Co=rng.standard_normal((n, nocc)),
                Cv=rng.standard_normal((n, nvir)), B=rng.standard_normal((nb, naux, nocc, nvir)))


def _check_grad(mol, seed, nb, nocc, nvir, what, atoms=None, **kw):
    x = _inputs(mol, seed, nb, nocc, nvir)
    ctx = ris_setup(mol, spherical=True, **kw)
    assert ctx.nao == orc.nao_sph(mol)
    gJ = ctx.grad_J(dev(x["D"]), dev(x["c"])).cpu().numpy()
    gK = ctx.grad_K(dev(x["Co"]), dev(x["Cv"]), dev(x["B"])).cpu().numpy()
    assert_parity(gJ, orc.grad_J_sph(mol, x["D"], x["c"], atoms=atoms)[0], what + " J")
    assert_parity(gK, orc.grad_K_sph(mol, x["Co"], x["Cv"], x["B"], atoms=atoms)[0], what + " K")
    return ctx, x, gJ, gK


@pytest.mark.parametrize("cfg", [1, 2])
def test_spherical_small_configs(cfg):
    wl = synth.make_workload(cfg)
    ctx, x, gJ, gK = _check_grad(wl.mol, 40 + cfg, 2, wl.nocc, wl.nvir, f"config {cfg} spherical")
    # host-buffer entry points take the spherical sizes too
    hJ = ctx.grad_J_host(x["D"], x["c"])
    hK = ctx.grad_K_host(x["Co"], x["Cv"], x["B"])
    assert np.abs(hJ - gJ).max() <= 5e-14 * np.abs(gJ).max() and np.abs(hK - gK).max() <= 5e-14 * np.abs(gK).max()
    ctx.close()


def test_spherical_all_classes_up_to_f():
    mol = synth.tiny_molecule(21, [[0, 1, 2, 3], [3, 2, 0], [1, 3], [0]],
                              [[0, 0, 0], [1.9, 0.4, -0.3], [-0.8, 1.7, 1.0], [0.5, -2.2, 1.4]], nprim=2)
    ctx, *_ = _check_grad(mol, 7, 6, 3, 5, "all classes spherical")
    assert all(ctx.npairs(la, lb) > 0 for la in range(4) for lb in range(la + 1))
    ctx.close()


def test_spherical_s_and_p_only_equals_cartesian_up_to_the_p_order():
    """s and p shells: the spherical functions ARE the Cartesian ones, p in the order y, z, x."""
    mol = synth.tiny_molecule(4, [[0, 1], [1, 0, 1], [0]], [[0, 0, 0], [1.7, 0.2, 0.4], [-0.9, 1.5, -0.6]])
    rng = np.random.default_rng(2)
    n = mol.nao
    D = rng.standard_normal((1, n, n))
    c = rng.standard_normal((1, mol.natoms))
    perm = []
    off = 0
    for l in mol.shell_l:
        perm += [off] if l == 0 else [off + 1, off + 2, off]       # spherical position k holds Cartesian component perm[k]
        off += 1 if l == 0 else 3
    perm = np.array(perm)
    Ds = D[:, perm][:, :, perm]
    c0, c1 = ris_setup(mol), ris_setup(mol, spherical=True)
    g0, g1 = c0.grad_J(dev(D), dev(c)).cpu().numpy(), c1.grad_J(dev(Ds), dev(c)).cpu().numpy()
    assert np.abs(g0 - g1).max() <= 5e-15 * np.abs(g0).max()
    c0.close(); c1.close()


def test_spherical_full_size_config5_sampled_atoms():
    """Config 5 (4s3p2d1f on 40 atoms: 1400 Cartesian / 1160 spherical AOs) at full size on sampled atoms."""
    wl = synth.make_workload(5)
    atoms = [0, 7, 19, 33]
    ctx, *_ = _check_grad(wl.mol, 55, 1, wl.nocc, wl.nvir, "config 5 spherical", atoms=atoms)
    ctx.close()


def test_spherical_fitting_step_and_matvec():
    """ris_fit_J / ris_fit_K / ris_resp_* with spherical inputs: v, T against the oracle's tensors transformed with U."""
    mol = synth.tiny_molecule(13, [[0, 2, 1], [3, 0], [2, 1]], [[0, 0, 0], [1.8, 0.3, -0.2], [-0.6, 1.6, 0.8]])
    x = _inputs(mol, 3, 2, 3, 4)
    U = orc.sph_matrix(mol)
    ctx = ris_setup(mol, spherical=True)
    v, cfit = ctx.fit_J(dev(x["D"]))
    v_ref, c_ref, _ = orc.fit_J(mol, orc.density_sph_to_cart(mol, x["D"]))
    assert_parity(v.cpu().numpy(), v_ref, "spherical v")
    cond = np.linalg.cond(orc.metric(mol))
    assert np.abs(cfit.cpu().numpy() - c_ref).max() <= 64 * cond * EPS * np.abs(c_ref).max()
    T, B = ctx.fit_K(dev(x["Co"]), dev(x["Cv"]))
    T_ref, B_ref = orc.fit_K(mol, U.T @ x["Co"], U.T @ x["Cv"])[:2]
    assert_parity(T.cpu().numpy(), T_ref, "spherical T")
    assert np.abs(B.cpu().numpy() - B_ref).max() <= 64 * cond * EPS * np.abs(B_ref).max()
    Q, _ = np.linalg.qr(np.random.default_rng(9).standard_normal((orc.nao_sph(mol), 7)))
    Co, Cv = np.ascontiguousarray(Q[:, :3]), np.ascontiguousarray(Q[:, 3:])
    X = np.random.default_rng(10).standard_normal((2, 3, 4))
    ctx.resp_setup(dev(Co), dev(Cv))
    got = ctx.resp_matvec(dev(X), 2.0, 0.25, 0.25).cpu().numpy()
    ref = orc.matvec_ris(mol, U.T @ Co, U.T @ Cv, X, 2.0, 0.25, 0.25)
    assert np.abs(got - ref).max() <= max(5e-14, 64 * cond * EPS) * np.abs(ref).max()
    ctx.close()


def test_spherical_combined_host_call_and_aux_ranges():
    """ris_grad_host (J + K + PQ from host buffers in one call) and the aux-range calls of the multi-GPU split with spherical
    inputs: the same boundary transformation serves every entry point."""
    wl = synth.make_workload(2)
    mol = wl.mol
    x = _inputs(mol, 77, 2, wl.nocc, wl.nvir)
    d_aux = np.random.default_rng(78).standard_normal((2, mol.natoms))
    ctx = ris_setup(mol, spherical=True)
    gJ = ctx.grad_J(dev(x["D"]), dev(x["c"])).cpu().numpy()
    gK = ctx.grad_K(dev(x["Co"]), dev(x["Cv"]), dev(x["B"])).cpu().numpy()
    gQ = ctx.grad_PQ(dev(x["c"]), dev(d_aux)).cpu().numpy()
    hJ, hK, hQ = ctx.grad_host(x["D"], x["c"], d_aux, x["Co"], x["Cv"], x["B"])
    for h, g in ((hJ, gJ), (hK, gK), (hQ, gQ)):
        assert np.abs(h - g).max() <= 5e-14 * np.abs(g).max()
    partJ = ctx.grad_J_range(dev(x["D"]), dev(x["c"]), 0, 13).cpu().numpy() + ctx.grad_J_range(dev(x["D"]), dev(x["c"]), 13, mol.natoms).cpu().numpy()
    partK = (ctx.grad_K_range(dev(x["Co"]), dev(x["Cv"]), dev(np.ascontiguousarray(x["B"][:, :13])), 0, 13).cpu().numpy()
             + ctx.grad_K_range(dev(x["Co"]), dev(x["Cv"]), dev(np.ascontiguousarray(x["B"][:, 13:])), 13, mol.natoms).cpu().numpy())
    assert np.abs(partJ - gJ).max() <= 5e-14 * np.abs(gJ).max()
    assert np.abs(partK - gK).max() <= 5e-14 * np.abs(gK).max()
    ctx.close()


def test_spherical_shapes_are_checked():
    mol = synth.tiny_molecule(4, [[0, 2], [1]], [[0, 0, 0], [1.7, 0.2, 0.4]])
    ctx = ris_setup(mol, spherical=True)
    assert ctx.nao == 1 + 5 + 3
    with pytest.raises((RisError, ValueError, AssertionError)):
        ctx.grad_J(dev(np.zeros((1, mol.nao, mol.nao))), dev(np.zeros((1, 2))))      # Cartesian-sized D is refused
    ctx.close()
