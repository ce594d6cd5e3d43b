"""The P-sharded step (SURVEY.md 8(e), NEXT-4a; paper_2511_18233_b200/shard.py) on the GPU: the range calls
ris_grad_J_range / ris_grad_K_range evaluated for every rank's share on ONE device must add up to the unsharded gradients
(real arithmetic, no collective), and -- when the box has two GPUs -- two NCCL ranks must each end up with them."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ris_oracle as orc
from paper_2511_18233_b200 import ris_setup, synth
from paper_2511_18233_b200.shard import aux_range, grad_JK_sharded

from test_gpu_parity import assert_parity, dev

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,world,jfit", [(2, 2, False), (2, 3, True), (3, 8, True)])
def test_sum_of_rank_shares_equals_the_unsharded_gradient(cfg, world, jfit):
    wl = synth.make_workload(cfg)
    mol = synth.with_jfit(wl.mol, cfg) if jfit else wl.mol
    rng = np.random.default_rng(70 + cfg)
    nbJ = wl.D.shape[0]
    c = rng.standard_normal((nbJ, synth.naux_jfit(mol)))
    ctx = ris_setup(mol, schwarz_tol=wl.schwarz_tol)
    D, cd, Co, Cv, B = dev(wl.D), dev(c), dev(wl.C_occ), dev(wl.C_vir), dev(wl.B)
    gJ, gK = ctx.grad_J(D, cd), ctx.grad_K(Co, Cv, B)
    sJ, sK = torch.zeros_like(gJ), torch.zeros_like(gK)
    for r in range(world):
        fr, pr = aux_range(ctx.naux_J, r, world), aux_range(ctx.naux, r, world)
        sJ += ctx.grad_J_range(D, cd, fr.start, fr.stop)
        sK += ctx.grad_K_range(Co, Cv, B[:, pr.start:pr.stop].contiguous(), pr.start, pr.stop)
    assert (sJ - gJ).abs().max().item() <= 5e-14 * gJ.abs().max().item()
    assert (sK - gK).abs().max().item() <= 5e-14 * gK.abs().max().item()
    if cfg == 2:            # and one share against the oracle's sum over the same aux functions
        pr = aux_range(ctx.naux, 1, world)
        part = ctx.grad_K_range(Co, Cv, B[:, pr.start:pr.stop].contiguous(), pr.start, pr.stop).cpu().numpy()
        ref, _ = orc.grad_K(mol, wl.C_occ, wl.C_vir, wl.B, aux=list(pr))
        assert_parity(part, ref, "K share of rank 1")
    # empty share
    z = ctx.grad_K_range(Co, Cv, B[:, :0].contiguous(), 5, 5)
    assert float(z.abs().max()) == 0.0
    ctx.close()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _nccl_worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world)
    try:
        wl = synth.make_workload(2)
        ctx = ris_setup(wl.mol)
        d = lambda x: torch.as_tensor(np.ascontiguousarray(x), dtype=torch.float64, device=f"cuda:{rank}")
        pr = aux_range(ctx.naux, rank, world)
        gJ, gK = grad_JK_sharded(ctx, d(wl.D), d(wl.c_aux), d(wl.C_occ), d(wl.C_vir), d(wl.B[:, pr.start:pr.stop]))
        fJ, fK = ctx.grad_J(d(wl.D), d(wl.c_aux)), ctx.grad_K(d(wl.C_occ), d(wl.C_vir), d(wl.B))
        out[rank] = bool((gJ - fJ).abs().max().item() <= 5e-14 * fJ.abs().max().item()
                         and (gK - fK).abs().max().item() <= 5e-14 * fK.abs().max().item())
        ctx.close()
    finally:
        dist.destroy_process_group()


def test_two_nccl_ranks_each_hold_the_full_gradient():
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (this pool's boxes expose one)")
    import torch.multiprocessing as mp
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_nccl_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    assert out[0] and out[1]
