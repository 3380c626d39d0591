"""Multi-GPU decomposition of the exchange apply: the TARGETS are sharded across ranks,
the occupied orbitals are replicated, every rank runs an independent exx_apply on its target block, and the
only collective is one all-reduce (sum) of n_tgt-sized energy data.  No data-path collective exists: every
(j,k) pair is independent (Eq. 1), and this is the paper's own suggestion (i) -- move orbitals,
not right-hand sides.  Host-side logic only; no method arithmetic.
"""
from __future__ import annotations

import torch


def shard_targets(n_tgt: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous block [k0, k1) of the n_tgt targets owned by `rank` (sizes differ by at most one)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside 0..world-1")
    base, rem = divmod(n_tgt, world)
    k0 = rank * base + min(rank, rem)
    return k0, k0 + base + (1 if rank < rem else 0)


def weak_scaling_targets(tgt_start: int, n_tgt: int, n_orb: int, rank: int) -> torch.Tensor:
    """bench.py's weak-scaling rule: rank r applies Vx to n_tgt targets starting at tgt_start + r*n_tgt,
    wrapping around the orbital set, so the per-GPU work is that of the single-GPU workload."""
    return (tgt_start + rank * n_tgt + torch.arange(n_tgt)) % n_orb


def reduce_energy(e_k_local: torch.Tensor, occ_tgt_local: torch.Tensor, k0: int, n_tgt: int, group=None):
    """All-reduce the per-target energies into the full [n_tgt] vector and E_x = 1/2 sum_k occ_k e_k: ONE collective
    over a buffer of n_tgt + 1 doubles (the energies in their slots, this rank's partial E_x in the last one).
    Works with any backend (nccl on GPUs, gloo in the CPU tests); a no-op without torch.distributed."""
    import torch.distributed as dist
    buf = torch.zeros(n_tgt + 1, dtype=torch.float64, device=e_k_local.device)
    buf[k0:k0 + e_k_local.numel()] = e_k_local
    buf[n_tgt] = 0.5 * torch.sum(occ_tgt_local * e_k_local)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
    return buf[:n_tgt], buf[n_tgt]


def shard_orbitals(n_orb: int, rank: int, world: int) -> tuple[int, int, int]:
    """Orbital block [j0, j1) held by `rank` at the start of the ring, and the common padded block length
    (blocks are padded with zero-occupation orbitals so every ring message has the same size)."""
    j0, j1 = shard_targets(n_orb, rank, world)
    return j0, j1, -(-n_orb // world) if n_orb else 0


def ring_apply(apply_block, psi_block: torch.Tensor, occ_block: torch.Tensor, rank: int, world: int, group=None):
    """Orbital ring of SURVEY.md 8(e) for orbitals that do not fit one GPU (the paper's suggestion (i),
    PAPER.md:285: move orbitals, not right-hand sides).

    Every rank keeps its targets and ONE block of occupied orbitals at a time; in `world` steps each block
    visits every rank.  Step s: start sending the held block to rank+1 and receiving the next one from rank-1
    (NCCL P2P over NVLink on GPUs, gloo in the CPU tests), call ``apply_block(psi, occ, accumulate=s > 0,
    last=s == world - 1)`` on the held block -- the transfer overlaps the compute -- then wait and swap.
    ``apply_block`` runs exx_apply with the plan's accumulate mode (exx_plan_set_accumulate), asking for the
    energy on the last step only.  psi_block [nb, ...] / occ_block [nb] must have the same (padded) shape on
    every rank; padding orbitals carry occ = 0 and contribute nothing.  Host logic only.
    """
    import torch.distributed as dist
    cur_psi, cur_occ = psi_block, occ_block
    nxt_psi, nxt_occ = torch.empty_like(psi_block), torch.empty_like(occ_block)
    for step in range(world):
        last = step == world - 1
        reqs = []
        if not last and world > 1:
            dst, src = (rank + 1) % world, (rank - 1) % world
            ops = [dist.P2POp(dist.isend, cur_psi, dst, group), dist.P2POp(dist.irecv, nxt_psi, src, group),
                   dist.P2POp(dist.isend, cur_occ, dst, group), dist.P2POp(dist.irecv, nxt_occ, src, group)]
            reqs = dist.batch_isend_irecv(ops)
        apply_block(cur_psi, cur_occ, accumulate=step > 0, last=last)
        for r in reqs:
            r.wait()
        if not last:
            cur_psi, nxt_psi = nxt_psi, cur_psi
            cur_occ, nxt_occ = nxt_occ, cur_occ
