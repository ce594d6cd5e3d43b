"""N > 1 path on CPU: world_size-2 (and 3) `gloo` processes exercise the state partition and the control-plane gather
of paper_2511_18233_b200/shard.py.  No GPU and no method arithmetic: each rank fills its block
with a function of the global state index, and the gathered result must be that function of 0..nstates-1."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2511_18233_b200.shard import gather_gradients, state_range


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
