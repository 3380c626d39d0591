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
