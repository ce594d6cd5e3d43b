"""N > 1 path on CPU: world_size-2 (and 3) `gloo` processes exercise the state partition and the control-plane gather
of paper_2511_18233_b200/shard.py.  No GPU and no method arithmetic: each rank fills its block
with a function of the global state index, and the gathered result must be that function of 0..nstates-1."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2511_18233_b200.shard import aux_range, gather_gradients, grad_JK_sharded, state_range


def test_state_range_partitions_exactly():
    for nstates in (0, 1, 2, 3, 5, 8, 17):
        for world in (1, 2, 3, 4, 8):
            seen = []
            for r in range(world):
                rg = state_range(nstates, r, world)
                seen += list(rg)
                assert len(rg) in (nstates // world, nstates // world + 1)
            assert seen == list(range(nstates))
    with pytest.raises(ValueError):
        state_range(3, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nstates, natoms, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = state_range(nstates, rank, world)
        local = torch.empty((len(mine), natoms, 3), dtype=torch.float64)
        for k, s in enumerate(mine):
            local[k] = s + 0.001 * torch.arange(natoms * 3, dtype=torch.float64).reshape(natoms, 3)
        full = gather_gradients(local, nstates)
        expect = torch.stack([s + 0.001 * torch.arange(natoms * 3, dtype=torch.float64).reshape(natoms, 3)
                              for s in range(nstates)]) if nstates else torch.empty((0, natoms, 3), dtype=torch.float64)
        out[rank] = bool(full.shape == expect.shape and torch.equal(full, expect))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,nstates", [(2, 5), (2, 1), (3, 3)])
def test_gather_over_gloo(world, nstates):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), nstates, 7, out), nprocs=world, join=True)
    assert all(out[r] for r in range(world)) and len(out) == world


def test_aux_range_partitions_exactly_in_lane_chunks():
    for naux in (0, 1, 20, 31, 32, 33, 40, 100, 300, 1200):
        for world in (1, 2, 3, 4, 8):
            seen = []
            for r in range(world):
                rg = aux_range(naux, r, world)
                seen += list(rg)
                if naux >= 32 * world and r < world - 1:
                    assert len(rg) % 32 == 0 and len(rg) > 0
            assert seen == list(range(naux)), (naux, world)
    assert [len(aux_range(300, r, 8)) for r in range(8)] == [64, 64, 32, 32, 32, 32, 32, 12]
    assert [len(aux_range(20, r, 8)) for r in range(8)] == [3, 3, 3, 3, 2, 2, 2, 2]


class _FakeCtx:
    """Stands in for RisContext in the CPU test of the sharded step's plumbing: the 'partial gradient' of a range is a
    known function of the aux indices in it, so the all-reduced sum over ranks is known in closed form."""

    def __init__(self, naux, naux_J, natoms):
        self.naux, self.naux_J, self.natoms = naux, naux_J, natoms

    def grad_J_range(self, D, c_aux, f_lo, f_hi, out):
        out.zero_()
        for f in range(f_lo, f_hi):
            out += c_aux[:, f].reshape(-1, 1, 1) * (f + 1)
        return out

    def grad_K_range(self, C_occ, C_vir, B_local, p_lo, p_hi, out):
        out.zero_()
        for k, P in enumerate(range(p_lo, p_hi)):
            out += B_local[:, k].sum(dim=(1, 2)).reshape(-1, 1, 1) * (P + 1)
        return out


def _worker_sharded(rank, world, port, naux, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        g = torch.Generator().manual_seed(5)
        nbJ, nbK, natoms, nocc, nvir = 2, 3, 4, 2, 3
        naux_J = 4 * naux
        D = torch.zeros((nbJ, 1, 1), dtype=torch.float64)
        c = torch.randn((nbJ, naux_J), dtype=torch.float64, generator=g)
        B = torch.randn((nbK, naux, nocc, nvir), dtype=torch.float64, generator=g)
        pr = aux_range(naux, rank, world)
        ctx = _FakeCtx(naux, naux_J, natoms)
        gJ, gK = grad_JK_sharded(ctx, D, c, None, None, B[:, pr.start:pr.stop].contiguous())
        wJ = torch.arange(1, naux_J + 1, dtype=torch.float64)
        wK = torch.arange(1, naux + 1, dtype=torch.float64)
        eJ = (c * wJ).sum(dim=1).reshape(-1, 1, 1).expand(nbJ, natoms, 3)
        eK = (B.sum(dim=(2, 3)) * wK).sum(dim=1).reshape(-1, 1, 1).expand(nbK, natoms, 3)
        ok = torch.allclose(gJ, eJ, rtol=1e-13, atol=1e-12) and torch.allclose(gK, eK, rtol=1e-13, atol=1e-12)
        bad = False
        try:
            grad_JK_sharded(ctx, D, c, None, None, B[:, : len(pr) + 1].contiguous()) if len(pr) + 1 <= naux else None
        except ValueError:
            bad = True
        out[rank] = bool(ok and (bad or len(pr) + 1 > naux))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,naux", [(2, 70), (2, 3), (3, 100)])
def test_sharded_step_plumbing_over_gloo(world, naux):
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker_sharded, args=(world, _free_port(), naux, out), nprocs=world, join=True)
    assert all(out[r] for r in range(world)) and len(out) == world
