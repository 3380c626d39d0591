"""The orbital ring of SURVEY.md 8(e) / NEXT-4 (PAPER.md:285 (i): move orbitals, not right-hand sides) on GPUs: one
process per GPU, NCCL point-to-point transfers of the orbital blocks, exx_apply with the plan's accumulate mode
(exx_plan_set_accumulate) on every block, the energies all-reduced at the end -- against the oracle's serial apply.

The NCCL case needs at least two GPUs; on a one-GPU box it is collected and skipped (NCCL refuses two ranks on one
device).  UNMEASURED ON HARDWARE in this repository's rounds: gpurun and the driver's round-end tiers give one GPU.

What a one-GPU box CAN run is the same worker with two ranks sharing cuda:0 over gloo: the orbital blocks travel between
the processes through host memory (gloo has no CUDA point-to-point), each rank uploads the block it holds and runs
exx_apply in accumulate mode on the GPU.  That executes the combination the NCCL world-2 case would -- the library's
kernels, accumulate mode, and a block that arrived from another rank -- minus NVLink.  The two ranks' kernels never
wait on one another (only the host processes do), so sharing the GPU cannot deadlock.  bench.py's whole multi-rank
branch is executed the same way (`--backend gloo`) at the end of this file."""
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


def _ring_worker(rank, world, port, out_dir, backend="nccl"):
    from paper_2501_16572_b200 import exx
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    gpu = rank if backend == "nccl" else 0                   # gloo: every rank on cuda:0
    torch.cuda.set_device(gpu)
    if backend == "nccl":
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", gpu))
    else:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda", gpu)
    blk_dev = dev if backend == "nccl" else torch.device("cpu")   # where the travelling orbital blocks live
    w = wl.scaled(wl.WORKLOADS[2], 7, 7, 0)                  # 48^3, 7 orbitals: blocks 4 + 3 (padded to 4) at world 2
    psi, _, _, _ = wl.make_inputs(w, "cpu")
    occ = torch.linspace(2.0, 0.2, w.n_orb, dtype=torch.float64)
    k0, k1 = sharding.shard_targets(w.n_tgt, rank, world)
    j0, j1, nb = sharding.shard_orbitals(w.n_orb, rank, world)
    psi_b = torch.zeros((nb,) + tuple(psi.shape[1:]), dtype=torch.float64, device=blk_dev)
    occ_b = torch.zeros(nb, dtype=torch.float64, device=blk_dev)
    psi_b[:j1 - j0] = psi[j0:j1].to(blk_dev)
    occ_b[:j1 - j0] = occ[j0:j1].to(blk_dev)
    my_tgt = psi[k0:k1].to(dev)
    my_occ_t = occ[k0:k1].to(dev)
    plan = exx.Plan.for_workload(w, max_batch=16, device=gpu)
    vx = torch.empty_like(my_tgt)
    result = {}

    def apply_block(p, o, accumulate, last):
        plan.set_accumulate(accumulate)
        _, e_k, _ = plan.apply(p.to(dev), o.to(dev), my_tgt, my_occ_t if last else None, vx=vx, n_c=8)
        if last:
            result["e_k"] = e_k
        torch.cuda.current_stream(dev).synchronize()         # the block may be overwritten by the next receive

    sharding.ring_apply(apply_block, psi_b, occ_b, rank, world)
    plan.set_accumulate(False)
    if backend == "nccl":
        e_all, ex = sharding.reduce_energy(result["e_k"], my_occ_t, k0, w.n_tgt)
    else:
        e_all, ex = sharding.reduce_energy(result["e_k"].cpu(), my_occ_t.cpu(), k0, w.n_tgt)
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
    _check_ring_against_oracle(tmp_path, world)


def _check_ring_against_oracle(tmp_path, world):
    w = wl.scaled(wl.WORKLOADS[2], 7, 7, 0)
    psi, _, _, _ = wl.make_inputs(w, "cpu")
    occ = np.linspace(2.0, 0.2, w.n_orb)
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    vx, e_k, ex = orc.exx_apply(plan, psi.numpy(), occ, psi.numpy(), occ)
    got = np.concatenate([np.load(tmp_path / f"ring_vx_{r}.npy") for r in range(world)])
    assert np.abs(got - vx).max() < TOL * np.abs(vx).max()
    assert np.abs(np.load(tmp_path / "ring_e.npy") - e_k).max() < TOL * np.abs(e_k).max()
    assert abs(np.load(tmp_path / "ring_ex.npy")[0] - ex) < TOL * abs(ex)


def test_orbital_ring_two_ranks_sharing_one_gpu_over_gloo(tmp_path):
    """Two ranks, both on cuda:0: blocks 4 + 3 (padded to 4) of 7 orbitals change hands once; every rank's vx block is
    accumulated from its own block and the one received from the other process."""
    import __graft_entry__ as ge
    ge.build()
    mp.spawn(_ring_worker, args=(2, _free_port(), str(tmp_path), "gloo"), nprocs=2, join=True)
    _check_ring_against_oracle(tmp_path, 2)


@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_bench_multi_rank_branch_on_one_gpu(scaling):
    """bench.py's N > 1 path end to end (process group, target sharding, the energy all-reduce inside the timed region,
    the max-over-ranks timing, the joint teardown, rank 0's instrumentation) with two ranks on this box's GPU
    (`--backend gloo`, a debug mode the line names), on config 1, whose E_x the oracle gives in seconds.  Weak scaling:
    rank r applies Vx to targets (r * 8 + 0..7) mod 8, i.e. both ranks to all 8 -- the union's E_x is twice the oracle's;
    strong scaling: 4 targets each -- exactly the oracle's."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(root, "bench.py"), "--gpus", "2", "--config", "1", "--steps", "3",
           "--warmup", "3", "--backend", "gloo", "--scaling", scaling, "--no-cpu-baseline", "--no-extras"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    d = json.loads(lines[0])
    w = wl.WORKLOADS[1]
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    _, _, ex = orc.exx_apply(plan, psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy())
    mult = 2 if scaling == "weak" else 1
    assert d["n_gpus"] == 2 and d["scaling"] == scaling and "gloo" in d["backend"]
    assert d["pair_solves_all_ranks"] == mult * w.pair_solves
    assert abs(d["E_x"] - mult * ex) < TOL * abs(mult * ex)
    assert d["value"] > 0 and d["gpu_launches"] > 0 and d["roofline"]["frac"] > 0
