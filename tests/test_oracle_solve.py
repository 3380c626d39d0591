"""Pins for the oracle's solve and apply (CPU only).

Ground truth independent of the Kronecker structure: the 3-D Laplacian is assembled here by brute
force (the stencil, with weights read from the textbook rationals in tests/golden, applied grid
point by grid point with wrap / truncation), and Eqs. 2-5 are evaluated on that dense
N x N matrix with LAPACK (solve / pinv / eigh / expm).  The oracle must reproduce them through
Eq. 7.
"""
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.linalg as sla

from oracle import exx_oracle as orc

P, D = orc.PERIODIC, orc.DIRICHLET


def _weights(golden_dir, order, h):
    with open(os.path.join(golden_dir, "fd_second_derivative_weights.txt")) as f:
        for line in f:
            p = line.split()
            if p and p[0] == str(order):
                return [float(Fraction(x)) / h ** 2 for x in p[1:]]
    raise KeyError(order)


def dense_laplacian(golden_dir, nx, ny, nz, h, bc, order):
    """L[idx(x,y,z), idx(x',y',z')], idx = x + nx*(y + ny*z), by applying the stencil point by point."""
    w = _weights(golden_dir, order, h)
    n0 = order // 2
    dims = (nx, ny, nz)
    N = nx * ny * nz
    L = np.zeros((N, N))
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                row = x + nx * (y + ny * z)
                for ax in range(3):
                    for q in range(-n0, n0 + 1):
                        c = [x, y, z]
                        c[ax] += q
                        if bc[ax] == P:
                            c[ax] %= dims[ax]
                        elif not (0 <= c[ax] < dims[ax]):
                            continue
                        L[row, c[0] + nx * (c[1] + ny * c[2])] += w[abs(q)]
    return L


CASES = [((8, 7, 6), (P, P, P)), ((6, 5, 9), (P, P, D)), ((5, 6, 7), (D, D, D)), ((4, 9, 5), (D, P, D))]


@pytest.mark.parametrize("dims,bc", CASES)
def test_unscreened_solve_matches_dense_direct_solve(dims, bc, golden_dir):
    nx, ny, nz = dims
    h = 0.4
    L = dense_laplacian(golden_dir, nx, ny, nz, h, bc, 12)
    assert np.allclose(L, L.T)
    plan = orc.make_plan(nx, ny, nz, h, bc, 12, 0.0)
    rng = np.random.default_rng(7)
    C = rng.standard_normal((3, nz, ny, nx))
    Y = orc.poisson_solve(plan, C)
    A = -L / (4 * np.pi)                        # Eq. 2: -(1/4pi) lap phi = rho
    for b in range(3):
        rho = C[b].ravel()
        if all(x == P for x in bc):
            phi = np.linalg.pinv(A, rcond=1e-12, hermitian=True) @ rho   # zero-mean solution; mean(rho) discarded (R3)
            assert abs(Y[b].mean()) < 1e-13 * np.abs(Y[b]).max()
        else:
            phi = np.linalg.solve(A, rho)
        assert np.allclose(Y[b].ravel(), phi, rtol=0, atol=2e-13 * np.abs(phi).max())
        # residual of the PDE itself
        res = A @ Y[b].ravel() - (rho - (rho.mean() if all(x == P for x in bc) else 0.0))
        assert np.abs(res).max() < 1e-12 * np.abs(rho).max()


@pytest.mark.parametrize("dims,bc", CASES)
def test_screened_solve_matches_dense_matrix_function(dims, bc, golden_dir):
    nx, ny, nz = dims
    h, omega = 0.4, 0.106
    L = dense_laplacian(golden_dir, nx, ny, nz, h, bc, 12)
    plan = orc.make_plan(nx, ny, nz, h, bc, 12, omega)
    rng = np.random.default_rng(11)
    C = rng.standard_normal((2, nz, ny, nx))
    Y = orc.poisson_solve(plan, C)
    # (a) eigh of the dense N x N matrix: no Kronecker structure used
    lam, U = np.linalg.eigh(L)
    mu = -lam
    f = np.where(np.abs(lam) < 1e-9, np.pi / omega ** 2,
                 4 * np.pi * (1 - np.exp(-np.where(np.abs(lam) < 1e-9, 1.0, mu) / (4 * omega ** 2)))
                 / np.where(np.abs(lam) < 1e-9, 1.0, mu))
    F = (U * f[None, :]) @ U.T
    for b in range(2):
        ref = F @ C[b].ravel()
        assert np.allclose(Y[b].ravel(), ref, rtol=0, atol=5e-13 * np.abs(ref).max())
    # (b) where L is invertible, the literal Eq. 5 (as read in R1): -4 pi L^-1 (I - expm(L/(4 w^2)))
    if not all(x == P for x in bc):
        F2 = -4 * np.pi * np.linalg.solve(L, np.eye(L.shape[0]) - sla.expm(L / (4 * omega ** 2)))
        ref = F2 @ C[0].ravel()
        assert np.allclose(Y[0].ravel(), ref, rtol=0, atol=1e-11 * np.abs(ref).max())


def test_plane_wave_analytic_solution(golden_dir):
    # rho = cos(2 pi mx x/Lx) cos(2 pi my y/Ly): an eigenfunction; phi = -4 pi / (lam_mx + lam_my + lam_0) rho
    nx, ny, nz, h = 16, 12, 10, 0.5
    w = _weights(golden_dir, 12, h)
    lam1 = lambda n, m: w[0] + 2 * sum(w[q] * np.cos(2 * np.pi * m * q / n) for q in range(1, 7))
    mx, my = 2, 3
    x = np.arange(nx)[None, None, :]
    y = np.arange(ny)[None, :, None]
    rho = np.cos(2 * np.pi * mx * x / nx) * np.cos(2 * np.pi * my * y / ny) * np.ones((nz, 1, 1))
    lam_sum = lam1(nx, mx) + lam1(ny, my) + lam1(nz, 0)
    for omega, mult in ((0.0, -4 * np.pi / lam_sum),
                        (0.106, -4 * np.pi / lam_sum * (1 - np.exp(lam_sum / (4 * 0.106 ** 2))))):
        plan = orc.make_plan(nx, ny, nz, h, (P, P, P), 12, omega)
        phi = orc.poisson_solve(plan, rho)
        assert np.allclose(phi, mult * rho, rtol=0, atol=1e-13 * abs(mult))
    # constant RHS: dropped for PBE0, scaled by pi/w^2 for HSE (reading R3)
    one = np.ones((nz, ny, nx))
    assert np.abs(orc.poisson_solve(orc.make_plan(nx, ny, nz, h, (P, P, P), 12, 0.0), one)).max() < 1e-12
    assert np.allclose(orc.poisson_solve(orc.make_plan(nx, ny, nz, h, (P, P, P), 12, 0.106), one),
                       np.pi / 0.106 ** 2, rtol=1e-12)


def test_vectorised_solve_equals_naive_loops():
    for bc, omega in (((P, P, P), 0.0), ((P, D, P), 0.106)):
        plan = orc.make_plan(5, 4, 6, 0.3, bc, 12, omega)
        c = np.random.default_rng(3).standard_normal((6, 4, 5))
        a = orc.poisson_solve(plan, c)
        b = orc.poisson_solve_loops(plan, c)
        assert np.allclose(a, b, rtol=0, atol=1e-13 * np.abs(b).max())


def test_eq8_per_slice_solve_equals_batch_solve_and_dense_function(golden_dir):
    """PAPER.md:74-78 (Eq. 8): the non-batch per-slice algorithm is the same linear map as the batch formalism
    (Eq. 11) and as the dense matrix function of the assembled Laplacian (Eq. 4) -- unequal axis lengths and mixed
    boundary conditions, so that a transposed slice or a swapped V1/V2 fails."""
    for dims, bc, omega in (((5, 4, 6), (P, P, P), 0.0), ((4, 6, 5), (P, D, P), 0.106), ((6, 5, 4), (D, P, D), 0.106)):
        nx, ny, nz = dims
        plan = orc.make_plan(nx, ny, nz, 0.3, bc, 12, omega)
        c = np.random.default_rng(8).standard_normal((nz, ny, nx))
        a = orc.poisson_solve_eq8(plan, c)
        assert np.allclose(a, orc.poisson_solve(plan, c), rtol=0, atol=1e-13 * np.abs(a).max())
        assert np.allclose(a, orc.poisson_solve_loops(plan, c), rtol=0, atol=1e-13 * np.abs(a).max())
        if omega == 0.0:
            continue
        # dense matrix function of the point-by-point assembled Laplacian (no Kronecker structure), screened kernel
        L = dense_laplacian(golden_dir, nx, ny, nz, 0.3, bc, 12)
        lam, U = np.linalg.eigh(L)
        small = np.abs(lam) < 1e-9
        mu = np.where(small, 1.0, -lam)
        f = np.where(small, np.pi / omega ** 2, 4 * np.pi * (1 - np.exp(-mu / (4 * omega ** 2))) / mu)
        ref = (U * f[None, :]) @ U.T @ c.ravel()
        assert np.allclose(a.ravel(), ref, rtol=0, atol=5e-12 * np.abs(ref).max())


def test_batch_invariance():
    # the batch formalism is the same linear map for any n_c and any batch composition
    plan = orc.make_plan(9, 8, 7, 0.3, (P, P, D), 12, 0.106)
    C = np.random.default_rng(5).standard_normal((7, 7, 8, 9))
    full = orc.poisson_solve(plan, C)
    for b in range(7):
        assert np.allclose(orc.poisson_solve(plan, C[b]), full[b], rtol=0, atol=1e-13 * np.abs(full).max())
    perm = np.array([3, 0, 6, 1, 5, 2, 4])
    assert np.allclose(orc.poisson_solve(plan, C[perm]), full[perm], rtol=0, atol=1e-13 * np.abs(full).max())


# ---- apply (Eq. 1 / Eq. 19b) -----------------------------------------------------------------

def _small_problem(seed=1, dims=(6, 5, 7), bc=(P, P, D), omega=0.106, n_occ=5, h=0.35):
    nx, ny, nz = dims
    plan = orc.make_plan(nx, ny, nz, h, bc, 12, omega)
    rng = np.random.default_rng(seed)
    psi = rng.standard_normal((n_occ, nz, ny, nx))
    occ = rng.uniform(0.1, 2.0, n_occ)
    return plan, psi, occ, rng


@pytest.mark.parametrize("bc,omega", [((P, P, P), 0.0), ((P, P, D), 0.106), ((P, P, P), 0.106)])
def test_apply_matches_dense_definition(bc, omega, golden_dir):
    plan, psi, occ, rng = _small_problem(bc=bc, omega=omega)
    nx, ny, nz, h = plan.nx, plan.ny, plan.nz, plan.h
    L = dense_laplacian(golden_dir, nx, ny, nz, h, bc, 12)
    lam, U = np.linalg.eigh(L)
    zero = np.abs(lam) < 1e-9
    mu = np.where(zero, 1.0, -lam)
    if omega > 0:
        f = np.where(zero, np.pi / omega ** 2, 4 * np.pi * (1 - np.exp(-mu / (4 * omega ** 2))) / mu)
    else:
        f = np.where(zero, 0.0, 4 * np.pi / mu)
    F = (U * f[None, :]) @ U.T
    tgt = rng.standard_normal((3, nz, ny, nx))
    occ_t = np.array([2.0, 0.7, 1e-13])
    vx, e_k, ex = orc.exx_apply(plan, psi, occ, tgt, occ_t, chunk=2)
    P_ = psi.reshape(len(occ), -1)
    for k in range(3):
        t = tgt[k].ravel()
        ref = np.zeros_like(t)
        for j in range(len(occ)):                      # Eq. 1, term by term
            ref -= occ[j] * P_[j] * (F @ (P_[j] * t))
        assert np.allclose(vx[k].ravel(), ref, rtol=0, atol=1e-12 * np.abs(ref).max())
        assert e_k[k] == pytest.approx(h ** 3 * t @ ref, rel=1e-11)
    assert ex == pytest.approx(0.5 * np.sum(occ_t * e_k), rel=1e-15)


def test_vx_is_hermitian_and_negative_semidefinite():
    plan, psi, occ, rng = _small_problem(seed=2)
    ab = rng.standard_normal((2,) + psi.shape[1:])
    vx, _, _ = orc.exx_apply(plan, psi, occ, ab)
    lhs = np.sum(ab[0] * vx[1])      # <a|Vx b>
    rhs = np.sum(ab[1] * vx[0])      # <b|Vx a>
    assert lhs == pytest.approx(rhs, rel=1e-12)
    # M = Psi^T W is Cholesky-factorisable up to sign (Eq. 20): -M is PSD
    W, _, _ = orc.exx_apply(plan, psi, occ, psi)
    M = psi.reshape(len(occ), -1) @ W.reshape(len(occ), -1).T
    assert np.allclose(M, M.T, rtol=0, atol=1e-12 * np.abs(M).max())
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).max() < 1e-12 * np.abs(M).max()


def test_linearity_in_occ_and_pair_symmetry():
    plan, psi, occ, rng = _small_problem(seed=4, bc=(P, P, P), omega=0.0)
    tgt = psi[:2]
    v1, _, _ = orc.exx_apply(plan, psi, occ, tgt)
    v2, _, _ = orc.exx_apply(plan, psi, 3.0 * occ, tgt)
    assert np.allclose(v2, 3.0 * v1, rtol=1e-13, atol=1e-13 * np.abs(v1).max())
    occ0 = occ.copy()
    occ0[1] = 0.0
    v3, _, _ = orc.exx_apply(plan, psi, occ0, tgt)
    v4, _, _ = orc.exx_apply(plan, np.delete(psi, 1, axis=0), np.delete(occ, 1), tgt)
    assert np.allclose(v3, v4, rtol=0, atol=1e-13 * np.abs(v3).max())
    # phi_jk = phi_kj
    a = orc.poisson_solve(plan, psi[0] * psi[3])
    b = orc.poisson_solve(plan, psi[3] * psi[0])
    assert np.array_equal(a, b)


def test_exchange_energy_double_loop_identity():
    # E_x = 1/2 sum_k occ_k <psi_k|Vx psi_k> = -1/2 sum_jk occ_j occ_k dV rho_jk^T f(L) rho_jk
    plan, psi, occ, rng = _small_problem(seed=6)
    _, e_k, ex = orc.exx_apply(plan, psi, occ, psi, occ)
    s = 0.0
    for j in range(len(occ)):
        for k in range(len(occ)):
            rho = psi[j] * psi[k]
            s += occ[j] * occ[k] * plan.dV * np.sum(rho * orc.poisson_solve(plan, rho))
    assert ex == pytest.approx(-0.5 * s, rel=1e-12)
    assert ex < 0
    assert np.all(e_k < 0)
