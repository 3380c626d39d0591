"""N > 1 path on CPU: world_size-2 gloo processes shard the targets, run the per-rank apply (here the
oracle stands in for the per-GPU exx_apply -- only the host-side decomposition is under test) and
all-reduce the energies; the result must equal the unsharded apply."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import exx_oracle as orc
from paper_2501_16572_b200 import sharding, workloads as wl


def test_shard_targets_partition():
    for n in (0, 1, 7, 64, 129):
        for world in (1, 2, 3, 8):
            blocks = [sharding.shard_targets(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n
            for a, b in zip(blocks, blocks[1:]):
                assert a[1] == b[0]
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_targets(4, 2, 2)
    idx = sharding.weak_scaling_targets(60, 8, 64, 1)
    assert idx.tolist() == [4, 5, 6, 7, 8, 9, 10, 11]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.set_num_threads(1)
    w = wl.scaled(wl.WORKLOADS[1], 6, 5, 1)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")          # replicated orbitals, same seed on every rank
    k0, k1 = sharding.shard_targets(w.n_tgt, rank, world)
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    vx, e_k, _ = orc.exx_apply(plan, psi.numpy(), occ.numpy(), tgt.numpy()[k0:k1], occ_t.numpy()[k0:k1])
    e_all, ex = sharding.reduce_energy(torch.from_numpy(e_k), occ_t[k0:k1], k0, w.n_tgt)
    np.save(os.path.join(out_dir, f"vx_{rank}.npy"), vx)
    if rank == 0:
        np.save(os.path.join(out_dir, "e_all.npy"), e_all.numpy())
        np.save(os.path.join(out_dir, "ex.npy"), np.array([float(ex)]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_target_sharding_matches_serial(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = wl.scaled(wl.WORKLOADS[1], 6, 5, 1)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    vx, e_k, ex = orc.exx_apply(plan, psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy())
    got = np.concatenate([np.load(tmp_path / f"vx_{r}.npy") for r in range(world)])
    assert np.array_equal(got, vx)                       # per-target columns are independent: bitwise equal
    assert np.allclose(np.load(tmp_path / "e_all.npy"), e_k, rtol=1e-15)
    assert np.load(tmp_path / "ex.npy")[0] == pytest.approx(ex, rel=1e-14)


def _ring_worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.set_num_threads(1)
    w = wl.scaled(wl.WORKLOADS[1], 7, 7, 0)                  # 7 orbitals over 3 ranks: blocks 3, 2, 2 (padded to 3)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    occ = torch.linspace(2.0, 0.2, w.n_orb, dtype=torch.float64)
    k0, k1 = sharding.shard_targets(w.n_tgt, rank, world)
    j0, j1, nb = sharding.shard_orbitals(w.n_orb, rank, world)
    psi_b = torch.zeros((nb,) + tuple(psi.shape[1:]), dtype=torch.float64)
    occ_b = torch.zeros(nb, dtype=torch.float64)
    psi_b[:j1 - j0] = psi[j0:j1]
    occ_b[:j1 - j0] = occ[j0:j1]
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    my_tgt = psi[k0:k1].numpy()
    vx = np.zeros_like(my_tgt)
    calls = []

    def apply_block(p, o, accumulate, last):                 # the oracle stands in for exx_apply + accumulate mode
        if not accumulate:
            vx[:] = 0.0
        for k in range(vx.shape[0]):
            orc.exx_accumulate(plan, p.numpy(), o.numpy(), my_tgt[k], vx[k])
        calls.append((accumulate, last))

    sharding.ring_apply(apply_block, psi_b, occ_b, rank, world)
    assert calls == [(s > 0, s == world - 1) for s in range(world)]
    np.save(os.path.join(out_dir, f"ring_vx_{rank}.npy"), vx)
    dist.barrier()
    dist.destroy_process_group()


def test_three_rank_orbital_ring_matches_serial(tmp_path):
    world = 3
    mp.spawn(_ring_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = wl.scaled(wl.WORKLOADS[1], 7, 7, 0)
    psi, _, _, _ = wl.make_inputs(w, "cpu")
    occ = np.linspace(2.0, 0.2, w.n_orb)
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    vx, _, _ = orc.exx_apply(plan, psi.numpy(), occ, psi.numpy())
    got = np.concatenate([np.load(tmp_path / f"ring_vx_{r}.npy") for r in range(world)])
    # each rank sums the orbital blocks in a different (rotated) order: equal to rounding, not bitwise
    assert np.abs(got - vx).max() < 1e-13 * np.abs(vx).max()


def test_shard_orbitals_padding():
    assert sharding.shard_orbitals(7, 0, 3) == (0, 3, 3)
    assert sharding.shard_orbitals(7, 2, 3) == (5, 7, 3)
    assert sharding.shard_orbitals(0, 0, 2) == (0, 0, 0)
