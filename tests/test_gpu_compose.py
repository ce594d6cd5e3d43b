"""The composed term <g^ris,(xi); {D1, D2}> / <g^ris,(xi); Gamma_IJ> (NEXT-1) assembled from the library calls
(paper_2511_18233_b200/compose.py, MO-factored form) against the oracle's AO-basis definition
(oracle.ris_oracle.ris_pair_scalar / ris_pair_gradient) -- two different algebraic routes to the same number.
Tolerance: the fitted quantities carry cond(M) eps (DESIGN.md R-cond)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import compose, ris_setup, synth

from test_gpu_parity import dev

pytestmark = pytest.mark.gpu
EPS = 2.220446049250313e-16


def _mol():
    return synth.tiny_molecule(31, [[0, 1, 2], [0, 1, 3], [0, 2]], [[0, 0, 0], [2.0, 0.3, -0.4], [-0.7, 1.8, 0.9]], nprim=2)


def test_pair_scalar_and_gradient_general_Y():
    mol = _mol()
    rng = np.random.default_rng(0)
    nmo = 9
    C = rng.standard_normal((mol.nao, nmo))
    Y1, Y2 = rng.standard_normal((2, nmo, nmo))
    D1, D2 = C @ Y1 @ C.T, C @ Y2 @ C.T
    ctx = ris_setup(mol)
    tol = 64.0 * np.linalg.cond(orc.metric(mol)) * EPS
    for cx in (0.0, 0.25):
        s = compose.ris_pair_scalar(ctx, dev(C), dev(Y1), dev(Y2), cx)
        s_ref = orc.ris_pair_scalar(mol, D1, D2, cx)
        g = compose.ris_pair_gradient(ctx, dev(C), dev(Y1), dev(Y2), cx).cpu().numpy()
        g_ref = orc.ris_pair_gradient(mol, D1, D2, cx)
        # scale: the J and K parts cancel partly, so measure against their separate sizes
        sJ = abs(orc.ris_pair_scalar(mol, D1, D2, 0.0)) + abs(s_ref)
        assert abs(s - s_ref) <= max(tol, 1e-12) * max(sJ, 1.0), (cx, s, s_ref)
        gs = np.abs(orc.ris_pair_gradient(mol, D1, D2, 0.0)).max() + np.abs(g_ref).max()
        assert np.abs(g - g_ref).max() <= max(tol, 1e-12) * gs, (cx, np.abs(g - g_ref).max(), gs)
    ctx.close()


def test_gamma_term_from_amplitudes():
    """Gamma_IJ = {R_I^S, R_J^S} + {L_I^A, L_J^A} from X, Y amplitudes (Eqs. 32-34) against the AO-basis oracle."""
    mol = _mol()
    rng = np.random.default_rng(1)
    nocc, nvir = 3, 5
    Co, Cv = rng.standard_normal((mol.nao, nocc)), rng.standard_normal((mol.nao, nvir))
    XI, YI, XJ, YJ = rng.standard_normal((4, nvir, nocc))
    cx = 0.25
    ctx = ris_setup(mol)
    g = compose.gamma_term_gradient(ctx, dev(Co), dev(Cv), dev(XI), dev(YI), dev(XJ), dev(YJ), cx).cpu().numpy()

    def ao(R, sign):
        U = Cv @ R @ Co.T
        return 0.5 * (U + sign * U.T)

    g_ref = orc.ris_pair_gradient(mol, ao(XI + YI, 1), ao(XJ + YJ, 1), cx) \
        + orc.ris_pair_gradient(mol, ao(XI - YI, -1), ao(XJ - YJ, -1), cx)
    tol = 64.0 * np.linalg.cond(orc.metric(mol)) * EPS
    gs = np.abs(orc.ris_pair_gradient(mol, ao(XI + YI, 1), ao(XJ + YJ, 1), 0.0)).max() + np.abs(g_ref).max()
    assert np.abs(g - g_ref).max() <= max(tol, 1e-12) * gs
    assert np.all(np.abs(g.sum(axis=0)) <= 1e-9 * np.abs(g).sum())
    ctx.close()
