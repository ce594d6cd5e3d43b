"""The seeded input generators reproduce the shapes SURVEY.md §8(a)/(d) lists for the five configs."""
import numpy as np
import pytest

from paper_2511_18233_b200 import synth

EXPECT = {1: (3, 25, 12), 2: (30, 300, 135), 3: (100, 1100, 480), 4: (300, 3000, 1350), 5: (40, 1400, 400)}


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_config_shapes(cfg):
    mol, _ = synth.make_molecule(cfg)
    assert (mol.natoms, mol.nao, mol.nshells) == EXPECT[cfg]
    d = np.linalg.norm(mol.coords[:, None] - mol.coords[None], axis=-1) + 10 * np.eye(mol.natoms)
    assert d.min() >= 0.96 * synth.ANGSTROM - 1e-9
    assert mol.aux_exponents.min() > 0.0173 and mol.aux_exponents.max() < 0.1557
    # x^l component of every shell has unit self-overlap
    for s in range(0, mol.nshells, max(1, mol.nshells // 17)):
        l = int(mol.shell_l[s]); o = int(mol.shell_prim_off[s]); n = int(mol.shell_nprim[s])
        a, dk = mol.prim_exp[o:o + n], mol.prim_coef[o:o + n]
        g = a[:, None] + a[None]
        S = (dk[:, None] * dk[None] * synth._dfact2(l) / (2 * g) ** l * (np.pi / g) ** 1.5).sum()
        assert abs(S - 1) < 1e-12


def test_workloads_are_reproducible_and_shaped():
    w = synth.make_workload(2)
    w2 = synth.make_workload(2)
    assert np.array_equal(w.B, w2.B) and np.array_equal(w.mol.coords, w2.mol.coords)
    assert w.D.shape == (2, 300, 300) and np.allclose(w.D[0], w.D[0].T) and not np.allclose(w.D[1], w.D[1].T)
    assert w.nvir == 2 * w.nocc and w.B.shape == (1, 30, w.nocc, w.nvir)
    w1 = synth.make_workload(1)
    assert (w1.nocc, w1.nvir) == (5, 20)
    w4 = synth.make_workload(4, with_B=False)
    assert (w4.nocc, w4.nvir) == (525, 1050) and w4.D.shape[0] == 3
    ext = w4.mol.coords[:, 0].max() - w4.mol.coords[:, 0].min()
    assert abs(ext / synth.ANGSTROM - 180.6) < 0.5
