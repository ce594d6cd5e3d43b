"""Multi-GPU: how the path shards.

The gradient of every state (excited state / state pair) is an independent problem: `ris_grad_J`, `ris_grad_K` and
`ris_grad_PQ` contract the same integrals with that state's D, c_aux, B.  So N GPUs = N processes, each with its own
`ris_setup` context on its own device (the packed pair data is replicated: <= 150 MB), each computing a contiguous
block of the states.  There is NO data-path collective: nothing is exchanged while the kernels run.  The only
communication is the control-plane gather of the finished `[nstates_local][natoms][3]` gradients (a few KB), for
which `torch.distributed` (NCCL on GPUs, gloo in the CPU tests) is plumbing.

This module holds only the index arithmetic and that gather; it performs none of the method's arithmetic.
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
