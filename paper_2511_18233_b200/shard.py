"""Multi-GPU: how the path shards.

The gradient of every state (excited state / state pair) is an independent problem: `ris_grad_J`, `ris_grad_K` and
`ris_grad_PQ` contract the same integrals with that state's D, c_aux, B.  So N GPUs = N processes, each with its own
`ris_setup` context on its own device (the packed pair data is replicated: <= 150 MB), each computing a contiguous
block of the states.  There is NO data-path collective: nothing is exchanged while the kernels run.  The only
communication is the control-plane gather of the finished `[nstates_local][natoms][3]` gradients (a few KB), for
which `torch.distributed` (NCCL on GPUs, gloo in the CPU tests) is plumbing.

Sharding ONE state over the auxiliary index (SURVEY.md 8(e), NEXT-4a): both three-centre contractions are sums over aux
functions, so rank r evaluates `ris_grad_J_range` / `ris_grad_K_range` on its block of them -- holding only its own slice
B[:, P_local] of the amplitudes-times-integrals tensor, the bulk of the input -- and ONE all-reduce of
`(nbatch_J + nbatch_K) natoms 3` doubles (NCCL over NVLink on GPUs; gloo in the CPU tests) completes both gradients on
every rank.  That all-reduce is the path's only exchange step; the two-centre term is a few microseconds and is
evaluated in full by every rank (identical, deterministic results).  Total work is fixed: strong scaling.

This module holds only the index arithmetic and the collectives; it performs none of the method's arithmetic.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def state_range(nstates: int, rank: int, world: int) -> range:
    """Contiguous block of states owned by `rank`: the first `nstates % world` ranks take one extra state.
    Ranks beyond the number of states own an empty range."""
    if nstates < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("state_range: bad arguments")
    q, r = divmod(nstates, world)
    lo = rank * q + min(rank, r)
    return range(lo, lo + q + (1 if rank < r else 0))


def gather_gradients(local: torch.Tensor, nstates: int, group=None) -> torch.Tensor:
    """All-gather the per-rank gradients `[len(state_range)][natoms][3]` into `[nstates][natoms][3]` on every rank
    (state order = rank order).  Ranks may own different numbers of states, including none."""
    world = dist.get_world_size(group)
    natoms = local.shape[1]
    counts = [len(state_range(nstates, r, world)) for r in range(world)]
    width = max(max(counts), 1)
    padded = torch.zeros((width, natoms, 3), dtype=local.dtype, device=local.device)
    padded[: local.shape[0]] = local
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    return torch.cat([p[:n] for p, n in zip(parts, counts)], dim=0)


def aux_range(naux: int, rank: int, world: int, align: int = 32) -> range:
    """Contiguous block of auxiliary functions owned by `rank`.  Blocks are multiples of `align` (the class kernels hand
    32 aux functions to the 32 lanes of a warp) while every rank still gets work; the last ranks take the ragged rest."""
    if naux < 0 or world < 1 or not (0 <= rank < world) or align < 1:
        raise ValueError("aux_range: bad arguments")
    units = -(-naux // align)                         # chunks of `align`
    if units < world:                                 # fewer chunks than ranks: fall back to single functions
        align, units = 1, naux
    q, r = divmod(units, world)
    lo_u = rank * q + min(rank, r)
    hi_u = lo_u + q + (1 if rank < r else 0)
    return range(min(lo_u * align, naux), min(hi_u * align, naux))


def grad_JK_sharded(ctx, D, c_aux, C_occ, C_vir, B_local, group=None, out=None):
    """One rank's part of the P-sharded step, then the all-reduce: returns (gJ, gK) complete on every rank.
    B_local [nbatch_K][len(aux_range(naux))][nocc][nvir] is this rank's slice of B; D, c_aux, C_occ, C_vir are replicated.
    `out` (optional): one preallocated [(nbatch_J + nbatch_K)][natoms][3] tensor that receives both results."""
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    nbJ, nbK = D.shape[0], B_local.shape[0]
    pr = aux_range(ctx.naux, rank, world)
    fr = aux_range(ctx.naux_J, rank, world)
    if B_local.shape[1] != len(pr):
        raise ValueError(f"B_local holds {B_local.shape[1]} aux functions, this rank owns {len(pr)}")
    if out is None:
        out = torch.empty((nbJ + nbK, ctx.natoms, 3), dtype=torch.float64, device=D.device)
    ctx.grad_J_range(D, c_aux, fr.start, fr.stop, out=out[:nbJ])
    ctx.grad_K_range(C_occ, C_vir, B_local, pr.start, pr.stop, out=out[nbJ:])
    dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)     # the one exchange step of the path
    return out[:nbJ], out[nbJ:]
