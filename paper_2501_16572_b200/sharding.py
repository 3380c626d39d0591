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
    """All-reduce the per-target energies into the full [n_tgt] vector and E_x = 1/2 sum_k occ_k e_k.
    Works with any backend (nccl on GPUs, gloo in the CPU tests); a no-op without torch.distributed."""
    import torch.distributed as dist
    e_k = torch.zeros(n_tgt, dtype=torch.float64, device=e_k_local.device)
    e_k[k0:k0 + e_k_local.numel()] = e_k_local
    ex = 0.5 * torch.sum(occ_tgt_local * e_k_local).reshape(1)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(e_k, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(ex, op=dist.ReduceOp.SUM, group=group)
    return e_k, ex[0]
