"""B200-native TDDFT-ris derivative-integral contractions (arxiv 2511.18233, Eq. 27).

    ctx = ris_setup(mol)                 # screening / sorting / packing on device
    gJ = ctx.grad_J(D, c_aux)            # [nbatch][natoms][3]
    gK = ctx.grad_K(C_occ, C_vir, B)
    gQ = ctx.grad_PQ(c_aux, d_aux)

The compute path is the CUDA library libris_b200.so (C ABI: include/ris.h); see DESIGN.md.
"""
from .ris import RisContext, RisError, RisOptions, load_library, probe_fp64_peak, ris_setup  # noqa: F401
