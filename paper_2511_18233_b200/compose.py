"""Caller-side assembly of the full TDDFT-ris term <g^ris,(xi); Gamma_IJ> from
the library calls.  Paper: Eqs. 5, 21-22 (kernel, index pairing), 25-27 (gradient / coupling expressions, derivative
of the RI-factorised integral), 32-34, 38-39 (Gamma_IJ, contraction notation).

For two AO matrices given in a common MO-like basis, D_i = C Y_i C^T (C [nao][nmo], Y_i [nmo][nmo]),
    S = <g^ris; {D1, D2}> = sum_AB M^-1_AB ( Tr[I^A D1] Tr[I^B D2] - c_x Tr[T^A Y2^T T^B Y1^T] ),   T^A = C^T I^A C,
and its derivative at fixed Y_i, C (Eq. 27) is
    G = G_J(D1, c2) + G_J(D2, c1) - G_PQ(c1, c2)                                   c_i = ris_fit_J(D_i)
        - c_x [ G_K(C, C, Z) - G_PQ_full(N) ],                                      (T, B) = ris_fit_K(C, C)
    Z^A = (Y2^T B^A Y1^T + Y1^T B^A Y2^T)^T,   N_CD = Tr[B^C Y2^T B^D Y1^T].
Every integral, its derivative, the metric solve and the AO <-> MO transforms of the three-index tensors run in the
library's CUDA kernels (ris_fit_J, ris_fit_K, ris_grad_J, ris_grad_K, ris_grad_PQ, ris_grad_PQ_full); what this module
adds is the MO-space bookkeeping between those calls -- products of [nmo][nmo] matrices, done with torch.matmul on the
device (plain library GEMMs).  It holds no arithmetic of the integral path and never touches the oracle.
"""
from __future__ import annotations

import torch


def ris_pair_scalar(ctx, C, Y1, Y2, c_x: float) -> float:
    """S = <g^ris; {C Y1 C^T, C Y2 C^T}> (device tensors, float64)."""
    D = torch.stack([C @ Y1 @ C.T, C @ Y2 @ C.T]).contiguous()
    v, c = ctx.fit_J(D)
    T, B = ctx.fit_K(C.contiguous(), C.contiguous())
    sk = torch.einsum("amn,anm->", T @ Y2.T, B @ Y1.T)
    return float(v[0] @ c[1] - c_x * sk)


def ris_pair_gradient(ctx, C, Y1, Y2, c_x: float) -> torch.Tensor:
    """[natoms][3]: d/dR of ris_pair_scalar at fixed C, Y1, Y2 (the <g^ris,(xi); {D1, D2}> of Eqs. 25-27)."""
    C = C.contiguous()
    D = torch.stack([C @ Y1 @ C.T, C @ Y2 @ C.T]).contiguous()
    _, c = ctx.fit_J(D)
    gJ = ctx.grad_J(D, torch.stack([c[1], c[0]]).contiguous()).sum(dim=0) - ctx.grad_PQ(c[0:1].contiguous(), c[1:2].contiguous())[0]
    if c_x == 0.0:
        return gJ
    _, B = ctx.fit_K(C, C)                                   # [naux][nmo][nmo]
    BY2, BY1 = B @ Y2.T, B @ Y1.T
    Z = Y2.T @ BY1 + Y1.T @ BY2                              # Z^A = Y2^T B^A Y1^T + Y1^T B^A Y2^T
    N = torch.einsum("cmn,dnm->cd", BY2, BY1)                # N_CD = Tr[B^C Y2^T B^D Y1^T]
    gK = ctx.grad_K(C, C, Z.transpose(1, 2).contiguous()[None])[0] - ctx.grad_PQ_full(N[None].contiguous())[0]
    return gJ - c_x * gK


def amplitudes_to_mo(R: torch.Tensor, sign: float) -> torch.Tensor:
    """MO-basis matrix of (1/2)(U + sign U^T), U = C_V R C_O^T (Eqs. 33-34), in the basis C = [C_O | C_V]:
    R [nvir][nocc]; sign = +1 for R^S, -1 for L^A."""
    nvir, nocc = R.shape
    Y = torch.zeros((nocc + nvir, nocc + nvir), dtype=R.dtype, device=R.device)
    Y[nocc:, :nocc] = 0.5 * R
    Y[:nocc, nocc:] = 0.5 * sign * R.T
    return Y


def gamma_term_gradient(ctx, C_occ, C_vir, X_I, Y_I, X_J, Y_J, c_x: float) -> torch.Tensor:
    """<g^ris,(xi); Gamma_IJ>, Gamma_IJ = {R_I^S, R_J^S} + {L_I^A, L_J^A}, R = X + Y, L = X - Y (Eqs. 32-34, 39);
    amplitudes [nvir][nocc].  I = J gives the excited-state-gradient term of Eq. 25, I != J the coupling term of Eq. 26
    (without the (E_J - E_I)^-1 factor, which is the caller's)."""
    C = torch.cat([C_occ, C_vir], dim=1).contiguous()
    g = ris_pair_gradient(ctx, C, amplitudes_to_mo(X_I + Y_I, 1.0), amplitudes_to_mo(X_J + Y_J, 1.0), c_x)
    return g + ris_pair_gradient(ctx, C, amplitudes_to_mo(X_I - Y_I, -1.0), amplitudes_to_mo(X_J - Y_J, -1.0), c_x)
