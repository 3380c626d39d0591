"""The orbital ring of SURVEY.md 8(e) / NEXT-4 (PAPER.md:285 (i): move orbitals, not right-hand sides) on GPUs: one
process per GPU, NCCL point-to-point transfers of the orbital blocks, exx_apply with the plan's accumulate mode
(exx_plan_set_accumulate) on every block, the energies all-reduced at the end -- against the oracle's serial apply.

Needs at least two GPUs; on a one-GPU box the test is collected and skipped (the same host logic runs on CPU with
gloo in tests/test_sharding_gloo.py).  UNMEASURED ON HARDWARE in this repository's rounds: gpurun and the driver's
round-end tiers give one GPU."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import exx_oracle as orc
from paper_2501_16572_b200 import sharding, workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _ring_worker(rank, world, port, out_dir):
    from paper_2501_16572_b200 import exx
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    dev = torch.device("cuda", rank)
    w = wl.scaled(wl.WORKLOADS[2], 7, 7, 0)                  # 48^3, 7 orbitals: blocks 4 + 3 (padded to 4) at world 2
    psi, _, _, _ = wl.make_inputs(w, "cpu")
    occ = torch.linspace(2.0, 0.2, w.n_orb, dtype=torch.float64)
    k0, k1 = sharding.shard_targets(w.n_tgt, rank, world)
    j0, j1, nb = sharding.shard_orbitals(w.n_orb, rank, world)
    psi_b = torch.zeros((nb,) + tuple(psi.shape[1:]), dtype=torch.float64, device=dev)
    occ_b = torch.zeros(nb, dtype=torch.float64, device=dev)
    psi_b[:j1 - j0] = psi[j0:j1].to(dev)
    occ_b[:j1 - j0] = occ[j0:j1].to(dev)
    my_tgt = psi[k0:k1].to(dev)
    my_occ_t = occ[k0:k1].to(dev)
    plan = exx.Plan.for_workload(w, max_batch=16, device=rank)
    vx = torch.empty_like(my_tgt)
    result = {}

    def apply_block(p, o, accumulate, last):
        plan.set_accumulate(accumulate)
        _, e_k, _ = plan.apply(p, o, my_tgt, my_occ_t if last else None, vx=vx, n_c=8)
        if last:
            result["e_k"] = e_k
        torch.cuda.current_stream(dev).synchronize()         # the block may be overwritten by the next receive

    sharding.ring_apply(apply_block, psi_b, occ_b, rank, world)
    plan.set_accumulate(False)
    e_all, ex = sharding.reduce_energy(result["e_k"], my_occ_t, k0, w.n_tgt)
    np.save(os.path.join(out_dir, f"ring_vx_{rank}.npy"), vx.cpu().numpy())
    if rank == 0:
        np.save(os.path.join(out_dir, "ring_e.npy"), e_all.cpu().numpy())
        np.save(os.path.join(out_dir, "ring_ex.npy"), np.array([float(ex)]))
    plan.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [1, pytest.param(2, marks=pytest.mark.skipif(
    torch.cuda.device_count() < 2, reason="the NCCL orbital ring needs at least two GPUs"))])
def test_orbital_ring_over_nccl_matches_oracle(tmp_path, world):
    """world = 1 runs the same worker (NCCL process group of one rank, accumulate mode, energy all-reduce) on a
    one-GPU box; world = 2 adds the P2P transfers."""
    import __graft_entry__ as ge
    ge.build()
    mp.spawn(_ring_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = wl.scaled(wl.WORKLOADS[2], 7, 7, 0)
    psi, _, _, _ = wl.make_inputs(w, "cpu")
    occ = np.linspace(2.0, 0.2, w.n_orb)
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    vx, e_k, ex = orc.exx_apply(plan, psi.numpy(), occ, psi.numpy(), occ)
    got = np.concatenate([np.load(tmp_path / f"ring_vx_{r}.npy") for r in range(world)])
    assert np.abs(got - vx).max() < TOL * np.abs(vx).max()
    assert np.abs(np.load(tmp_path / "ring_e.npy") - e_k).max() < TOL * np.abs(e_k).max()
    assert abs(np.load(tmp_path / "ring_ex.npy")[0] - ex) < TOL * abs(ex)
