"""Thin Python binding of the C ABI in include/ris.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libris_b200.so; PyTorch is used for device
memory and streams.  There is no CPU path: if the shared library is missing or no CUDA device is
usable, calls raise RisError.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# RIS_B200_LIB: load a side-by-side variant build (paper_2511_18233_b200.build with RIS_BUILD_TAG) instead -- kernel tuning only
LIB_PATH = os.environ.get("RIS_B200_LIB") or os.path.join(_HERE, "libris_b200.so")
_lib = None

EXPORTS = [
    "ris_setup", "ris_grad_J", "ris_grad_K", "ris_grad_PQ", "ris_grad_J_host", "ris_grad_K_host", "ris_grad_PQ_host", "ris_grad_host",
    "ris_fit_J", "ris_metric", "ris_fit_K", "ris_grad_PQ_full", "ris_set_jfit", "ris_naux_J", "ris_metric_J",
    "ris_resp_setup", "ris_resp_matvec", "ris_resp_free", "ris_grad_K_range", "ris_grad_J_range",
    "ris_destroy", "ris_strerror", "ris_nao", "ris_naux", "ris_natoms", "ris_npairs", "ris_npairs_total",
    "ris_nprimpairs", "ris_ntriplets", "ris_ntriplets_unscreened", "ris_npair_elements", "ris_p_batch",
    "ris_profile_reset", "ris_profile_enable", "ris_profile_count", "ris_profile_get", "ris_profile_get_work",
    # include/ris_bench.h: measurement / diagnostics, not the product boundary
    "ris_probe_fp64_peak", "ris_probe_fp64_mma_peak", "ris_diag_gemm2_layout",
]


class RisError(RuntimeError):
    pass


class RisOptions(C.Structure):
    _fields_ = [("schwarz_tol", C.c_double), ("deterministic", C.c_int), ("p_batch", C.c_int), ("profile", C.c_int),
                ("spherical", C.c_int)]


def load_library():
    """dlopen libris_b200.so (built in-tree by paper_2511_18233_b200.build).  Fails loudly when absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RisError(f"{LIB_PATH} not found: build it with `python -m paper_2511_18233_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, ci, cd = C.c_void_p, C.c_int, C.c_double
    lib.ris_setup.argtypes = [C.POINTER(vp), ci, vp, ci, vp, vp, vp, vp, vp, vp, vp, C.POINTER(RisOptions), vp]
    lib.ris_grad_J.argtypes = [vp, ci, vp, vp, vp]
    lib.ris_grad_K.argtypes = [vp, ci, ci, ci, vp, vp, vp, vp]
    lib.ris_grad_PQ.argtypes = [vp, ci, vp, vp, vp]
    lib.ris_grad_K_range.argtypes = [vp, ci, ci, ci, vp, vp, vp, ci, ci, vp]
    lib.ris_grad_J_range.argtypes = [vp, ci, vp, vp, ci, ci, vp]
    lib.ris_fit_J.argtypes = [vp, ci, vp, vp, vp]
    lib.ris_metric.argtypes = [vp, vp]
    lib.ris_metric_J.argtypes = [vp, vp]
    lib.ris_set_jfit.argtypes = [vp, ci, vp, vp, vp]
    lib.ris_resp_setup.argtypes = [vp, ci, ci, vp, vp]
    lib.ris_resp_matvec.argtypes = [vp, ci, cd, cd, cd, vp, vp]
    lib.ris_resp_free.argtypes = [vp]
    lib.ris_fit_K.argtypes = [vp, ci, ci, vp, vp, vp, vp]
    lib.ris_grad_PQ_full.argtypes = [vp, ci, vp, vp]
    lib.ris_grad_J_host.argtypes = [vp, ci, vp, vp, vp]
    lib.ris_grad_K_host.argtypes = [vp, ci, ci, ci, vp, vp, vp, vp]
    lib.ris_grad_PQ_host.argtypes = [vp, ci, vp, vp, vp]
    lib.ris_grad_host.argtypes = [vp, ci, vp, vp, vp, ci, ci, ci, vp, vp, vp, vp, vp, vp]
    lib.ris_destroy.argtypes = [vp]
    lib.ris_strerror.argtypes = [ci]
    lib.ris_strerror.restype = C.c_char_p
    for name in ("ris_nao", "ris_naux", "ris_naux_J", "ris_natoms", "ris_p_batch", "ris_profile_reset", "ris_profile_count"):
        getattr(lib, name).argtypes = [vp]
    lib.ris_profile_enable.argtypes = [vp, ci]
    for name in ("ris_npairs", "ris_nprimpairs"):
        getattr(lib, name).argtypes = [vp, ci, ci]
        getattr(lib, name).restype = C.c_longlong
    for name in ("ris_npairs_total", "ris_ntriplets", "ris_ntriplets_unscreened", "ris_npair_elements"):
        getattr(lib, name).argtypes = [vp]
        getattr(lib, name).restype = C.c_longlong
    lib.ris_profile_get.argtypes = [vp, ci, C.POINTER(C.c_char_p), C.POINTER(C.c_float)]
    lib.ris_profile_get_work.argtypes = [vp, ci, C.POINTER(cd), C.POINTER(cd)]
    lib.ris_probe_fp64_peak.argtypes = [C.POINTER(cd), vp]
    lib.ris_probe_fp64_mma_peak.argtypes = [C.POINTER(cd), vp]
    lib.ris_diag_gemm2_layout.argtypes = [vp, vp, C.POINTER(ci), C.POINTER(ci), C.POINTER(ci), C.POINTER(ci)]
    _lib = lib
    return lib


def _check(rc: int):
    if rc != 0:
        raise RisError(f"ris error {rc}: {load_library().ris_strerror(rc).decode()}")


def _np(x, dt):
    return np.ascontiguousarray(x, dtype=dt)


def probe_fp64_peak() -> float:
    """Achieved TFLOP/s of an independent-DFMA-chain kernel on the current device."""
    import torch
    if not torch.cuda.is_available():
        raise RisError("no CUDA device")
    out = C.c_double()
    _check(load_library().ris_probe_fp64_peak(C.byref(out), C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return out.value


def probe_fp64_mma_peak() -> float:
    """Achieved TFLOP/s of independent mma.sync f64 chains on the current device."""
    import torch
    if not torch.cuda.is_available():
        raise RisError("no CUDA device")
    out = C.c_double()
    _check(load_library().ris_probe_fp64_mma_peak(C.byref(out), C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return out.value


class RisContext:
    """ris_setup(coords, shells, aux_exponents) -> context with ris_grad_J / ris_grad_K / ris_grad_PQ."""

    def __init__(self, mol, *, schwarz_tol: float = 1e-13, deterministic: bool = False, p_batch: int = 0,
                 profile: bool = False, spherical: bool = False, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RisError("no CUDA device: the ris library has no CPU fallback")
        self._lib = load_library()
        self._torch = torch
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.device = torch.device("cuda", torch.cuda.current_device())
        arrs = (_np(mol.coords, np.float64), _np(mol.shell_atom, np.int32), _np(mol.shell_l, np.int32),
                _np(mol.shell_nprim, np.int32), _np(mol.shell_prim_off, np.int32), _np(mol.prim_exp, np.float64),
                _np(mol.prim_coef, np.float64), _np(mol.aux_exponents, np.float64))
        opt = RisOptions(schwarz_tol, int(deterministic), int(p_batch), int(profile), int(spherical))
        h = C.c_void_p()
        _check(self._lib.ris_setup(C.byref(h), arrs[0].shape[0], arrs[0].ctypes.data, arrs[1].shape[0],
                                   arrs[1].ctypes.data, arrs[2].ctypes.data, arrs[3].ctypes.data, arrs[4].ctypes.data,
                                   arrs[5].ctypes.data, arrs[6].ctypes.data, arrs[7].ctypes.data, C.byref(opt),
                                   C.c_void_p(self.stream.cuda_stream)))
        self._h = h
        self.nao = self._lib.ris_nao(h)            # AOs of the caller's basis (spherical: sum of 2l+1)
        self.nao_cart = int(sum((int(l) + 1) * (int(l) + 2) // 2 for l in arrs[2]))
        self.naux = self._lib.ris_naux(h)
        self.natoms = self._lib.ris_natoms(h)
        self.naux_J = self._lib.ris_naux_J(h)
        if getattr(mol, "jfit", None) is not None:
            self.set_jfit(*mol.jfit)

    def set_jfit(self, aux_atom, aux_l, aux_exp):
        """J-fit auxiliary set with p functions (ris_set_jfit): shells (atom, l in {0, 1}, exponent); the J-type calls then
        take naux_J coefficients per state."""
        at, ll, ex = _np(aux_atom, np.int32), _np(aux_l, np.int32), _np(aux_exp, np.float64)
        if not (at.shape == ll.shape == ex.shape and at.ndim == 1):
            raise RisError("set_jfit: aux_atom, aux_l, aux_exp must be 1-D arrays of one length")
        with self._ordered():
            _check(self._lib.ris_set_jfit(self._h, at.shape[0], at.ctypes.data, ll.ctypes.data, ex.ctypes.data))
        self.naux_J = self._lib.ris_naux_J(self._h)

    # ---- stream ordering: the library enqueues on the stream given at setup.  When the caller's CURRENT torch stream
    # is a different one (where its inputs were produced and where it will read the outputs), the setup stream first
    # waits for the current stream and the current stream afterwards waits for the setup stream.
    class _Ordered:
        def __init__(self, ctx):
            self.ctx = ctx

        def __enter__(self):
            torch = self.ctx._torch
            self.cur = torch.cuda.current_stream(self.ctx.device)
            if self.cur != self.ctx.stream:
                self.ctx.stream.wait_stream(self.cur)

        def __exit__(self, *exc):
            if self.cur != self.ctx.stream:
                self.cur.wait_stream(self.ctx.stream)

    def _ordered(self):
        return RisContext._Ordered(self)

    # ---- queries
    def npairs(self, la, lb):
        return int(self._lib.ris_npairs(self._h, la, lb))

    def nprimpairs(self, la, lb):
        return int(self._lib.ris_nprimpairs(self._h, la, lb))

    @property
    def npairs_total(self):
        return int(self._lib.ris_npairs_total(self._h))

    @property
    def ntriplets(self):
        return int(self._lib.ris_ntriplets(self._h))

    @property
    def ntriplets_unscreened(self):
        return int(self._lib.ris_ntriplets_unscreened(self._h))

    @property
    def npair_elements(self):
        return int(self._lib.ris_npair_elements(self._h))

    @property
    def p_batch(self):
        return int(self._lib.ris_p_batch(self._h))

    # ---- device-pointer calls (torch CUDA tensors, float64, contiguous)
    def _dev(self, t, shape):
        torch = self._torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise RisError("expected a contiguous float64 CUDA tensor")
        if tuple(t.shape) != tuple(shape):
            raise RisError(f"shape {tuple(t.shape)} != expected {tuple(shape)}")
        return C.c_void_p(t.data_ptr())

    def grad_J(self, D, c_aux, out=None):
        nb = D.shape[0]
        if out is None:
            out = self._torch.empty((nb, self.natoms, 3), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_grad_J(self._h, nb, self._dev(D, (nb, self.nao, self.nao)),
                                        self._dev(c_aux, (nb, self.naux_J)), self._dev(out, (nb, self.natoms, 3))))
        return out

    def grad_K(self, C_occ, C_vir, B, out=None):
        nb, nocc, nvir = B.shape[0], C_occ.shape[1], C_vir.shape[1]
        if out is None:
            out = self._torch.empty((nb, self.natoms, 3), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_grad_K(self._h, nb, nocc, nvir, self._dev(C_occ, (self.nao, nocc)),
                                        self._dev(C_vir, (self.nao, nvir)), self._dev(B, (nb, self.naux, nocc, nvir)),
                                        self._dev(out, (nb, self.natoms, 3))))
        return out

    def grad_K_range(self, C_occ, C_vir, B_local, p_lo, p_hi, out=None):
        """Partial K-type gradient over aux functions [p_lo, p_hi); B_local holds only that range."""
        nb, nocc, nvir = B_local.shape[0], C_occ.shape[1], C_vir.shape[1]
        if out is None:
            out = self._torch.empty((nb, self.natoms, 3), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_grad_K_range(self._h, nb, nocc, nvir, self._dev(C_occ, (self.nao, nocc)),
                                              self._dev(C_vir, (self.nao, nvir)),
                                              self._dev(B_local, (nb, p_hi - p_lo, nocc, nvir)), int(p_lo), int(p_hi),
                                              self._dev(out, (nb, self.natoms, 3))))
        return out

    def grad_J_range(self, D, c_aux, f_lo, f_hi, out=None):
        """Partial J-type gradient over J-fit functions [f_lo, f_hi)."""
        nb = D.shape[0]
        if out is None:
            out = self._torch.empty((nb, self.natoms, 3), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_grad_J_range(self._h, nb, self._dev(D, (nb, self.nao, self.nao)),
                                              self._dev(c_aux, (nb, self.naux_J)), int(f_lo), int(f_hi),
                                              self._dev(out, (nb, self.natoms, 3))))
        return out

    def grad_PQ(self, c_aux, d_aux, out=None):
        nb = c_aux.shape[0]
        if out is None:
            out = self._torch.empty((nb, self.natoms, 3), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_grad_PQ(self._h, nb, self._dev(c_aux, (nb, self.naux_J)), self._dev(d_aux, (nb, self.naux_J)),
                                         self._dev(out, (nb, self.natoms, 3))))
        return out

    # ---- fitting step, J type (argument marshalling only)
    def fit_J(self, D):
        """(v, c): v[s][P] = sum D^s_{mu nu} (mu nu|P), c = M^-1 v; both [nbatch][naux_J] on the device."""
        nb = D.shape[0]
        v = self._torch.empty((nb, self.naux_J), dtype=self._torch.float64, device=self.device)
        c = self._torch.empty((nb, self.naux_J), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_fit_J(self._h, nb, self._dev(D, (nb, self.nao, self.nao)), self._dev(v, (nb, self.naux_J)),
                                       self._dev(c, (nb, self.naux_J))))
        return v, c

    def fit_K(self, C_occ, C_vir):
        """(T, B): T[P][i][a] = sum C_occ[mu,i] (mu nu|P) C_vir[nu,a], B = M^-1 T; both on the device."""
        nocc, nvir = C_occ.shape[1], C_vir.shape[1]
        T = self._torch.empty((self.naux, nocc, nvir), dtype=self._torch.float64, device=self.device)
        B = self._torch.empty((self.naux, nocc, nvir), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_fit_K(self._h, nocc, nvir, self._dev(C_occ, (self.nao, nocc)), self._dev(C_vir, (self.nao, nvir)),
                                       self._dev(T, (self.naux, nocc, nvir)), self._dev(B, (self.naux, nocc, nvir))))
        return T, B

    def grad_PQ_full(self, G, out=None):
        nb = G.shape[0]
        if out is None:
            out = self._torch.empty((nb, self.natoms, 3), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_grad_PQ_full(self._h, nb, self._dev(G, (nb, self.naux, self.naux)),
                                              self._dev(out, (nb, self.natoms, 3))))
        return out

    def metric(self):
        M = self._torch.empty((self.naux, self.naux), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_metric(self._h, self._dev(M, (self.naux, self.naux))))
        return M

    def metric_J(self):
        n = self.naux_J
        M = self._torch.empty((n, n), dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_metric_J(self._h, self._dev(M, (n, n))))
        return M

    # ---- coupling-matrix products (excitation-energy stage, ris Z-vector)
    def resp_setup(self, C_occ, C_vir):
        nocc, nvir = C_occ.shape[1], C_vir.shape[1]
        with self._ordered():
            _check(self._lib.ris_resp_setup(self._h, nocc, nvir, self._dev(C_occ, (self.nao, nocc)), self._dev(C_vir, (self.nao, nvir))))
        self._resp_shape = (nocc, nvir)

    def resp_matvec(self, X, cJ, cKA, cKB, out=None):
        """sigma[v][i][a] = sum_jb [cJ (ia|jb) - cKA (ij|ab) - cKB (ib|ja)]^ris X[v][j][b]"""
        shape = getattr(self, "_resp_shape", None)
        if shape is None:
            raise RisError("resp_matvec before resp_setup")
        nvec = X.shape[0]
        if out is None:
            out = self._torch.empty((nvec,) + shape, dtype=self._torch.float64, device=self.device)
        with self._ordered():
            _check(self._lib.ris_resp_matvec(self._h, nvec, float(cJ), float(cKA), float(cKB), self._dev(X, (nvec,) + shape),
                                             self._dev(out, (nvec,) + shape)))
        return out

    def resp_free(self):
        _check(self._lib.ris_resp_free(self._h))
        self._resp_shape = None

    # ---- host-buffer calls (numpy arrays or CPU tensors, float64, C-contiguous; copies happen inside the C call)
    @staticmethod
    def _host(x, what="input"):
        """(pointer, shape, keep-alive).  float64 and C-contiguous are REQUIRED of tensors and of numpy arrays alike: a silent
        conversion copy would make the C call read (or, for outputs, fill) a temporary."""
        if hasattr(x, "data_ptr"):
            import torch
            if x.is_cuda or not x.is_contiguous() or x.dtype != torch.float64:
                raise RisError(f"{what}: expected a contiguous float64 CPU tensor, got {x.dtype} on {x.device}")
            return C.c_void_p(x.data_ptr()), tuple(x.shape), x
        a = np.asarray(x)
        if a.dtype != np.float64 or not a.flags.c_contiguous:
            raise RisError(f"{what}: expected a C-contiguous float64 array, got dtype {a.dtype}, "
                           f"c_contiguous={a.flags.c_contiguous}")
        return C.c_void_p(a.ctypes.data), a.shape, a

    @staticmethod
    def _shape(p, shape, what):
        """Host buffers carry no size across the C ABI: a wrong shape would be read (or written) out of bounds."""
        if tuple(p[1]) != tuple(shape):
            raise RisError(f"{what}: shape {tuple(p[1])} != expected {tuple(shape)}")

    def _host_out(self, out, shape):
        if out is None:
            out = np.empty(shape)
        p = self._host(out, "out")
        if tuple(p[1]) != tuple(shape):
            raise RisError(f"out: shape {tuple(p[1])} != expected {tuple(shape)}")
        return out, p

    def grad_J_host(self, D, c_aux, out=None):
        pD, pc = self._host(D, "D"), self._host(c_aux, "c_aux")
        nb = pD[1][0]
        self._shape(pD, (nb, self.nao, self.nao), "D"); self._shape(pc, (nb, self.naux_J), "c_aux")
        out, po = self._host_out(out, (nb, self.natoms, 3))
        with self._ordered():
            _check(self._lib.ris_grad_J_host(self._h, nb, pD[0], pc[0], po[0]))
        return out

    def grad_K_host(self, C_occ, C_vir, B, out=None):
        po, pv, pB = self._host(C_occ, "C_occ"), self._host(C_vir, "C_vir"), self._host(B, "B")
        nb, nocc, nvir = pB[1][0], po[1][1], pv[1][1]
        self._shape(po, (self.nao, nocc), "C_occ"); self._shape(pv, (self.nao, nvir), "C_vir")
        self._shape(pB, (nb, self.naux, nocc, nvir), "B")
        out, pg = self._host_out(out, (nb, self.natoms, 3))
        with self._ordered():
            _check(self._lib.ris_grad_K_host(self._h, nb, nocc, nvir, po[0], pv[0], pB[0], pg[0]))
        return out

    def grad_PQ_host(self, c_aux, d_aux, out=None):
        pc, pd = self._host(c_aux, "c_aux"), self._host(d_aux, "d_aux")
        nb = pc[1][0]
        self._shape(pc, (nb, self.naux_J), "c_aux"); self._shape(pd, (nb, self.naux_J), "d_aux")
        out, pg = self._host_out(out, (nb, self.natoms, 3))
        with self._ordered():
            _check(self._lib.ris_grad_PQ_host(self._h, nb, pc[0], pd[0], pg[0]))
        return out

    def grad_host(self, D, c_aux, d_aux, C_occ, C_vir, B, out=None):
        """(gJ, gK, gPQ) from host buffers in one call (H2D of B overlapped with the kernels)."""
        pD, pc, pd = self._host(D, "D"), self._host(c_aux, "c_aux"), self._host(d_aux, "d_aux")
        po, pv, pB = self._host(C_occ, "C_occ"), self._host(C_vir, "C_vir"), self._host(B, "B")
        nbJ, nbK, nocc, nvir = pD[1][0], pB[1][0], po[1][1], pv[1][1]
        self._shape(pD, (nbJ, self.nao, self.nao), "D"); self._shape(pc, (nbJ, self.naux_J), "c_aux")
        self._shape(pd, (nbJ, self.naux_J), "d_aux"); self._shape(po, (self.nao, nocc), "C_occ")
        self._shape(pv, (self.nao, nvir), "C_vir"); self._shape(pB, (nbK, self.naux, nocc, nvir), "B")
        if out is None:
            out = (None, None, None)
        oJ, pJ = self._host_out(out[0], (nbJ, self.natoms, 3))
        oK, pK = self._host_out(out[1], (nbK, self.natoms, 3))
        oQ, pQ = self._host_out(out[2], (nbJ, self.natoms, 3))
        with self._ordered():
            _check(self._lib.ris_grad_host(self._h, nbJ, pD[0], pc[0], pd[0], nbK, nocc, nvir, po[0], pv[0], pB[0],
                                           pJ[0], pK[0], pQ[0]))
        return oJ, oK, oQ

    # ---- measurement / diagnostics (include/ris_bench.h)
    def gemm2_layout(self):
        """(ao_pos[nao], panel_rows, tile_cols, ntiles, novf) of the pair-restricted Gamma^P GEMM-2."""
        pos = np.empty(self.nao_cart, dtype=np.int32)
        r, c, nt, nv = C.c_int(), C.c_int(), C.c_int(), C.c_int()
        _check(self._lib.ris_diag_gemm2_layout(self._h, pos.ctypes.data, C.byref(r), C.byref(c), C.byref(nt), C.byref(nv)))
        return pos, r.value, c.value, nt.value, nv.value

    # ---- profiling
    def profile_reset(self):
        _check(self._lib.ris_profile_reset(self._h))

    def profile_enable(self, on: bool):
        _check(self._lib.ris_profile_enable(self._h, int(bool(on))))

    def profile(self):
        """[(kernel name, ms, algorithmic flops, algorithmic bytes)] for every launch since the last reset
        (needs profile=True)."""
        self.stream.synchronize()
        n = self._lib.ris_profile_count(self._h)
        out = []
        for i in range(n):
            name, ms, fl, by = C.c_char_p(), C.c_float(), C.c_double(), C.c_double()
            _check(self._lib.ris_profile_get(self._h, i, C.byref(name), C.byref(ms)))
            _check(self._lib.ris_profile_get_work(self._h, i, C.byref(fl), C.byref(by)))
            out.append((name.value.decode(), ms.value, fl.value, by.value))
        return out

    def close(self):
        if getattr(self, "_h", None):
            self._lib.ris_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def ris_setup(mol, **kw) -> RisContext:
    return RisContext(mol, **kw)
