"""Seeded synthetic workloads: the five BASELINE.json configs.

This module is shared by the tests, bench.py and smoke(); it holds NONE of the method's
arithmetic (no FD matrices, no solves, no exchange sums) -- only the input generators:
seeded Gaussian noise, a separable Gaussian low-pass, a slab envelope, Cholesky-QR
orthonormalisation under the h^3 weight and Fermi-Dirac occupations.  It imports neither the
CUDA extension nor ``oracle``.

The inputs stand in for the paper's Mo-bulk / TiO2-slab orbitals, which need
SPARC, pseudopotentials and atomic structures that do not exist here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import numpy as np
import torch

PERIODIC = 0
DIRICHLET = 1
BASE_SEED = 20250116


@dataclass(frozen=True)
class Workload:
    name: str
    cfg: int              # 1-based index into BASELINE.json:configs
    nx: int
    ny: int
    nz: int
    h: float
    bc: tuple             # per axis (x, y, z)
    order: int
    omega: float          # <= 0: unscreened
    n_orb: int
    tgt_start: int
    n_tgt: int
    smooth_sigma: float   # grid points; 0 = raw noise
    envelope_sigma: float  # bohr; 0 = none (slab confinement along z)
    fermi: bool           # Fermi-Dirac occupations, else all 2.0
    default_nc: int

    @property
    def N(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def seed(self) -> int:
        return BASE_SEED + self.cfg

    @property
    def pair_solves(self) -> int:
        return self.n_orb * self.n_tgt

    @property
    def flops_per_solve(self) -> float:
        # algorithmic: six mode products, 2*N*n flops each; padding not credited
        return 4.0 * self.N * (self.nx + self.ny + self.nz)


P, D = PERIODIC, DIRICHLET
WORKLOADS = {
    1: Workload("cfg1_tiny_16c_pbe0", 1, 16, 16, 16, 0.5, (P, P, P), 12, 0.0, 8, 0, 8, 0.0, 0.0, False, 64),
    2: Workload("cfg2_bulk_48c_hse", 2, 48, 48, 48, 0.25, (P, P, P), 12, 0.106, 64, 0, 64, 2.0, 0.0, False, 1024),
    3: Workload("cfg3_slab_60x60x120_hse", 3, 60, 60, 120, 0.25, (P, P, D), 12, 0.106, 256, 0, 256, 2.0, 8.0, True, 1024),
    4: Workload("cfg4_metal_96c_hse", 4, 96, 96, 96, 0.2, (P, P, P), 12, 0.106, 1536, 896, 256, 2.0, 0.0, True, 512),
    5: Workload("cfg5_metal_120c_hse", 5, 120, 120, 120, 0.2, (P, P, P), 12, 0.106, 3200, 2176, 128, 2.0, 0.0, True, 256),
}


def scaled(w: Workload, n_orb: int, n_tgt: int | None = None, tgt_start: int | None = None) -> Workload:
    """Same grid/operator with fewer orbitals (parity sub-cases and bounded CPU samples)."""
    n_tgt = min(n_orb, w.n_tgt) if n_tgt is None else n_tgt
    tgt_start = min(w.tgt_start, n_orb - n_tgt) if tgt_start is None else tgt_start
    return replace(w, n_orb=n_orb, n_tgt=n_tgt, tgt_start=tgt_start)


def occupations(w: Workload) -> np.ndarray:
    """occ = 2.0, or Fermi-Dirac 2/(1+exp((e_i-mu)/kT)) with e_i evenly spaced in [-0.5, 0.5] Ha,
    mu = 0.2 Ha, kT = 0.01 Ha (BASELINE.json configs 3-5)."""
    n = w.n_orb
    if not w.fermi:
        return np.full(n, 2.0)
    e = -0.5 + np.arange(n, dtype=np.float64) / max(n - 1, 1)
    return 2.0 / (1.0 + np.exp((e - 0.2) / 0.01))


def _gauss_taps(sigma: float):
    r = int(round(4 * sigma))
    d = np.arange(-r, r + 1, dtype=np.float64)
    k = np.exp(-d * d / (2 * sigma * sigma))
    return r, k / k.sum()


def _smooth_axis(x: torch.Tensor, dim: int, sigma: float, circular: bool) -> torch.Tensor:
    r, k = _gauss_taps(sigma)
    out = torch.zeros_like(x)
    n = x.shape[dim]
    for t, d in zip(k.tolist(), range(-r, r + 1)):
        if circular:
            out.add_(torch.roll(x, shifts=d, dims=dim), alpha=t)
        else:  # zero padding beyond the box
            if d >= 0:
                if d < n:
                    out.narrow(dim, d, n - d).add_(x.narrow(dim, 0, n - d), alpha=t)
            elif -d < n:
                out.narrow(dim, 0, n + d).add_(x.narrow(dim, -d, n + d), alpha=t)
    return out


def _cholqr_(psi2d: torch.Tensor, dV: float, col_chunk: int = 1 << 18) -> None:
    """In-place Cholesky-QR: rows of psi2d [n, N] become orthonormal under the weight dV."""
    G = (psi2d @ psi2d.T) * dV
    L = torch.linalg.cholesky(G)
    N = psi2d.shape[1]
    for c0 in range(0, N, col_chunk):
        c1 = min(N, c0 + col_chunk)
        psi2d[:, c0:c1] = torch.linalg.solve_triangular(L, psi2d[:, c0:c1], upper=False)


def make_orbitals(w: Workload, device: str | torch.device = "cpu", orb_chunk: int = 64) -> torch.Tensor:
    """[n_orb, nz, ny, nx] FP64 orbitals, dV * Psi Psi^T = I.

    Noise is drawn per orbital chunk from a generator seeded ``w.seed`` on ``device`` (numpy
    default_rng on the host, torch Philox on CUDA: the two devices give different -- each
    deterministic -- data; whoever generates hands the same bytes to both the oracle and the GPU).
    """
    device = torch.device(device)
    n, shape = w.n_orb, (w.nz, w.ny, w.nx)
    psi = torch.empty((n, *shape), dtype=torch.float64, device=device)
    if device.type == "cpu":
        rng = np.random.default_rng(w.seed)
        gen = None
    else:
        gen = torch.Generator(device=device)
        gen.manual_seed(w.seed)
    if w.envelope_sigma > 0:
        z = (torch.arange(w.nz, dtype=torch.float64, device=device) + 1.0) * w.h
        z0 = (w.nz + 1) * w.h / 2.0
        env = torch.exp(-(z - z0) ** 2 / (2.0 * w.envelope_sigma ** 2))[None, :, None, None]
    for j0 in range(0, n, orb_chunk):
        j1 = min(n, j0 + orb_chunk)
        if gen is None:
            x = torch.from_numpy(rng.standard_normal((j1 - j0, *shape)))
        else:
            x = torch.randn((j1 - j0, *shape), dtype=torch.float64, device=device, generator=gen)
        if w.smooth_sigma > 0:
            x = _smooth_axis(x, 3, w.smooth_sigma, w.bc[0] == PERIODIC)
            x = _smooth_axis(x, 2, w.smooth_sigma, w.bc[1] == PERIODIC)
            x = _smooth_axis(x, 1, w.smooth_sigma, w.bc[2] == PERIODIC)
        if w.envelope_sigma > 0:
            x = x * env
        psi[j0:j1] = x
    flat = psi.view(n, -1)
    dV = w.h ** 3
    _cholqr_(flat, dV)
    _cholqr_(flat, dV)   # second pass (CholeskyQR2) restores orthonormality to rounding
    return psi


def make_inputs(w: Workload, device: str | torch.device = "cpu"):
    """(psi [n_orb,...], occ [n_orb], tgt view [n_tgt,...] into psi, occ_tgt [n_tgt])."""
    psi = make_orbitals(w, device)
    occ = torch.from_numpy(occupations(w)).to(psi.device)
    tgt = psi[w.tgt_start:w.tgt_start + w.n_tgt]
    occ_tgt = occ[w.tgt_start:w.tgt_start + w.n_tgt]
    return psi, occ, tgt, occ_tgt


def make_complex_orbitals(w: Workload, device: str | torch.device = "cpu") -> torch.Tensor:
    """[n_orb, 2, nz, ny, nx] complex orbitals as two real planes for the Bloch-periodic variant: real part = the
    workload's orbitals, imaginary part = half of the previous orbital (deterministic; data only, no arithmetic of
    the method)."""
    re = make_orbitals(w, device)
    return torch.stack([re, 0.5 * torch.roll(re, shifts=1, dims=0)], dim=1).contiguous()


def make_rhs(w: Workload, n_rhs: int, device: str | torch.device = "cpu", seed_offset: int = 1000) -> torch.Tensor:
    """[n_rhs, nz, ny, nx] seeded N(0,1) right-hand sides for the bare solver (Fig. 1-style sweeps)."""
    device = torch.device(device)
    shape = (n_rhs, w.nz, w.ny, w.nx)
    if device.type == "cpu":
        return torch.from_numpy(np.random.default_rng(w.seed + seed_offset).standard_normal(shape))
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed + seed_offset)
    return torch.randn(shape, dtype=torch.float64, device=device, generator=gen)
