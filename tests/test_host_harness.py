"""CPU checks of the CUDA path's arithmetic without a GPU: the generated per-class recurrences and the
Boys interpolation (paper_2511_18233_b200/csrc) are compiled as plain C++ by tests/host_harness and
compared with the oracle and with mpmath.  Test-only: the product has no CPU path."""
import ctypes as C
import math
import os
import subprocess

import mpmath
import numpy as np
import pytest

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import synth
from paper_2511_18233_b200.csrc import gen_classes

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(ROOT, "paper_2511_18233_b200", "csrc")


@pytest.fixture(scope="module")
def harness():
    gen_classes.main()
    so = os.path.join(HERE, "host_harness", "libharness.so")
    src = os.path.join(HERE, "host_harness", "harness.cpp")
    deps = [src, os.path.join(CSRC, "ris_core.cuh"), os.path.join(CSRC, "ris_boys_table.h"),
            os.path.join(CSRC, "generated", "ris_classes.cuh")]
    if not os.path.exists(so) or any(os.path.getmtime(d) > os.path.getmtime(so) for d in deps):
        subprocess.check_call(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-I", CSRC,
                               "-o", so, src])
    lib = C.CDLL(so)
    lib.harness_boys.argtypes = [C.c_int, C.c_double, C.c_void_p]
    lib.harness_triplet.argtypes = [C.c_int, C.c_int, C.c_int] + [C.c_void_p] * 4 + [C.c_double, C.c_double,
                                                                                    C.c_void_p, C.c_int, C.c_void_p]
    lib.harness_triplet0.argtypes = lib.harness_triplet.argtypes
    lib.harness_triplet_aux.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int] + [C.c_void_p] * 4 + [C.c_double, C.c_double,
                                                                                                 C.c_void_p, C.c_int, C.c_void_p]
    lib.harness_triplet0_aux.argtypes = lib.harness_triplet_aux.argtypes
    return lib


@pytest.mark.parametrize("M", [0, 1, 2, 3, 4, 5, 6, 7, 8])
def test_device_boys_interpolation_vs_mpmath(harness, M):
    mpmath.mp.dps = 40
    rng = np.random.default_rng(M)
    Ts = np.concatenate([[0.0, 1e-12, 1.0 / 64, 1.0 / 64 + 1e-9, 0.5, 39.98, 39.9999, 40.0, 40.0001, 55.0, 88.0, 150.0, 1e4],
                         rng.uniform(0, 40, 300), rng.uniform(40, 100, 50)])
    F = np.zeros(M + 1)
    worst = 0.0
    for T in Ts:
        harness.harness_boys(M, float(T), F.ctypes.data)
        for m in range(M + 1):
            ref = 1.0 / (2 * m + 1) if T == 0 else float(mpmath.gammainc(m + 0.5, 0, T) / (2 * mpmath.mpf(T) ** (m + 0.5)))
            worst = max(worst, abs(F[m] - ref) / ref)
    assert worst < 2e-14, worst


CLASSES = [(0, 0), (1, 0), (1, 1), (2, 0), (2, 1), (2, 2), (3, 0), (3, 1), (3, 2), (3, 3)]


@pytest.mark.parametrize("la,lb,span", [(la, lb, "normal") for la, lb in CLASSES] +
                         [(la, lb, "extreme") for la, lb in CLASSES])
def test_class_recurrence_vs_oracle(harness, la, lb, span):
    """One contracted triplet per class: VRR + accumulation + HRR (or the direct step on the s centre of an (l,s) pair) +
    derivative + contraction against the oracle's McMurchie-Davidson result (a different algorithm), for near and far aux
    centres.  span = "extreme": exponents log-uniform in [0.05, 300] (ratios up to 6000 inside one pair: the product
    centre sits on top of either centre) -- what the two-host rule and the direct step exist for."""
    rng = np.random.default_rng(10 * la + lb)
    lo, hi = (0.15, 4.0) if span == "normal" else (0.05, 300.0)
    for trial, dist in enumerate([1.5, 6.0, 40.0]):
        coords = np.array([[0.1, -0.2, 0.3], [1.1, 0.7, -0.6], [0, 0, 0]], dtype=float)
        v = rng.normal(size=3)
        coords[2] = coords[0] + dist * v / np.linalg.norm(v)
        mol = synth.tiny_molecule(100 + trial, [[la], [lb], []], coords, lo=lo, hi=hi, nprim=3)
        nca, ncb = synth.ncart(la), synth.ncart(lb)
        nb = 2
        tile = rng.standard_normal((nb, nca, ncb))
        G = np.zeros((nb, mol.nao, mol.nao))
        G[:, :nca, nca:] = tile
        P = 2
        g, _ = orc.grad_J(mol, G, np.eye(3)[P][None].repeat(nb, 0))
        # primitive-pair records exactly as ris_setup packs them
        A, B = coords[0], coords[1]
        prim = []
        for ka in range(3):
            for kb in range(3):
                a, b = mol.prim_exp[ka], mol.prim_exp[3 + kb]
                p = a + b
                # P - host centre; (l,s) pairs are hosted on the l shell whatever the exponents (ris_setup.cuh)
                PZ = -(b / p) * (A - B) if (a >= b or lb == 0) else (a / p) * (A - B)
                Kab = math.exp(-a * b / p * np.dot(A - B, A - B))
                coef = mol.prim_coef[ka] * mol.prim_coef[3 + kb] * Kab * 2 * math.pi ** 2.5 / p
                prim.append([p, PZ[0], PZ[1], PZ[2], 0.5 / p, 2 * a, 2 * b, coef])
        prim = np.ascontiguousarray(prim)
        alpha = mol.aux_exponents[P]
        auxfac = (2 * alpha / math.pi) ** 0.75 / alpha
        out = np.zeros((nb, 6))
        AB = A - B
        Cc = np.ascontiguousarray(coords[P])
        rc = harness.harness_triplet(la, lb, 9, prim.ctypes.data, A.ctypes.data, AB.ctypes.data, Cc.ctypes.data,
                                     alpha, auxfac, np.ascontiguousarray(tile).ctypes.data, nb, out.ctypes.data)
        assert rc == 0
        ref = np.concatenate([g[:, 0, :], g[:, 1, :]], axis=1)
        scale = np.abs(ref).max()
        np.testing.assert_allclose(out, ref, rtol=0, atol=2e-13 * scale)
        # translational invariance closes the aux centre
        np.testing.assert_allclose(-(out[:, :3] + out[:, 3:]), g[:, 2, :], rtol=0, atol=2e-13 * scale)


@pytest.mark.parametrize("la,lb", CLASSES)
def test_undifferentiated_class_recurrence_vs_oracle(harness, la, lb):
    """Fitting step (NEXT-1): one contracted triplet per class, sum_ab tile_ab (ab|P), against the oracle's v_P."""
    rng = np.random.default_rng(50 + 10 * la + lb)
    for trial, dist in enumerate([1.5, 6.0, 40.0]):
        coords = np.array([[0.1, -0.2, 0.3], [1.1, 0.7, -0.6], [0, 0, 0]], dtype=float)
        v = rng.normal(size=3)
        coords[2] = coords[0] + dist * v / np.linalg.norm(v)
        mol = synth.tiny_molecule(200 + trial, [[la], [lb], []], coords, lo=0.15, hi=4.0, nprim=3)
        nca, ncb = synth.ncart(la), synth.ncart(lb)
        nb = 2
        tile = rng.standard_normal((nb, nca, ncb))
        G = np.zeros((nb, mol.nao, mol.nao))
        G[:, :nca, nca:] = tile
        P = 2
        ref = orc.vec_J(mol, G)[:, P]
        A, B = coords[0], coords[1]
        prim = []
        for ka in range(3):
            for kb in range(3):
                a, b = mol.prim_exp[ka], mol.prim_exp[3 + kb]
                p = a + b
                PZ = -(b / p) * (A - B) if (a >= b or lb == 0) else (a / p) * (A - B)
                Kab = math.exp(-a * b / p * np.dot(A - B, A - B))
                coef = mol.prim_coef[ka] * mol.prim_coef[3 + kb] * Kab * 2 * math.pi ** 2.5 / p
                prim.append([p, PZ[0], PZ[1], PZ[2], 0.5 / p, 2 * a, 2 * b, coef])
        prim = np.ascontiguousarray(prim)
        alpha = mol.aux_exponents[P]
        auxfac = (2 * alpha / math.pi) ** 0.75 / alpha
        out = np.zeros(nb)
        AB = A - B
        Cc = np.ascontiguousarray(coords[P])
        rc = harness.harness_triplet0(la, lb, 9, prim.ctypes.data, A.ctypes.data, AB.ctypes.data, Cc.ctypes.data,
                                      alpha, auxfac, np.ascontiguousarray(tile).ctypes.data, nb, out.ctypes.data)
        assert rc == 0
        np.testing.assert_allclose(out, ref, rtol=0, atol=2e-13 * max(np.abs(ref).max(), 1e-3))


def _prim_records(mol, A, B, lb):
    """primitive-pair records exactly as ris_setup packs them (3 primitives per shell)"""
    prim = []
    for ka in range(3):
        for kb in range(3):
            a, b = mol.prim_exp[ka], mol.prim_exp[3 + kb]
            p = a + b
            PZ = -(b / p) * (A - B) if (a >= b or lb == 0) else (a / p) * (A - B)
            Kab = math.exp(-a * b / p * np.dot(A - B, A - B))
            coef = mol.prim_coef[ka] * mol.prim_coef[3 + kb] * Kab * 2 * math.pi ** 2.5 / p
            prim.append([p, PZ[0], PZ[1], PZ[2], 0.5 / p, 2 * a, 2 * b, coef])
    return np.ascontiguousarray(prim)


@pytest.mark.parametrize("la,lb", CLASSES)
def test_p_aux_class_recurrence_vs_oracle(harness, la, lb):
    """NEXT-2: a p-type auxiliary shell on the third centre.  Derivative and undifferentiated contracted
    triplets of every class, each p component, against the oracle's Hermite-shift evaluation (a different algorithm: the
    CUDA path takes one Obara-Saika step on the aux centre)."""
    rng = np.random.default_rng(300 + 10 * la + lb)
    for trial, dist in enumerate([1.3, 5.0, 35.0]):
        coords = np.array([[0.1, -0.2, 0.3], [1.1, 0.7, -0.6], [0, 0, 0]], dtype=float)
        v = rng.normal(size=3)
        coords[2] = coords[0] + dist * v / np.linalg.norm(v)
        mol = synth.tiny_molecule(400 + trial, [[la], [lb], []], coords, lo=0.15, hi=6.0, nprim=3)
        alpha = float(rng.uniform(0.1, 1.5))
        mol.jfit = (np.array([2]), np.array([1]), np.array([alpha]))
        nca, ncb = synth.ncart(la), synth.ncart(lb)
        nb = 2
        tile = rng.standard_normal((nb, nca, ncb))
        G = np.zeros((nb, mol.nao, mol.nao))
        G[:, :nca, nca:] = tile
        A, B = coords[0], coords[1]
        prim = _prim_records(mol, A, B, lb)
        auxfac = (2 * alpha / math.pi) ** 0.75 * 2.0 * math.sqrt(alpha) / alpha
        AB = A - B
        Cc = np.ascontiguousarray(coords[2])
        v_ref = orc.vec_J(mol, G)                        # [nb][3]
        for comp in range(3):
            g, _ = orc.grad_J(mol, G, np.eye(3)[comp][None].repeat(nb, 0))
            out = np.zeros((nb, 6))
            rc = harness.harness_triplet_aux(la, lb, comp + 1, 9, prim.ctypes.data, A.ctypes.data, AB.ctypes.data, Cc.ctypes.data,
                                             alpha, auxfac, np.ascontiguousarray(tile).ctypes.data, nb, out.ctypes.data)
            assert rc == 0
            ref = np.concatenate([g[:, 0, :], g[:, 1, :]], axis=1)
            scale = np.abs(g).max()
            np.testing.assert_allclose(out, ref, rtol=0, atol=2e-13 * scale)
            np.testing.assert_allclose(-(out[:, :3] + out[:, 3:]), g[:, 2, :], rtol=0, atol=2e-13 * scale)
            out0 = np.zeros(nb)
            rc = harness.harness_triplet0_aux(la, lb, comp + 1, 9, prim.ctypes.data, A.ctypes.data, AB.ctypes.data,
                                              Cc.ctypes.data, alpha, auxfac, np.ascontiguousarray(tile).ctypes.data, nb,
                                              out0.ctypes.data)
            assert rc == 0
            np.testing.assert_allclose(out0, v_ref[:, comp], rtol=0, atol=2e-13 * max(np.abs(v_ref).max(), 1e-3))
