"""Pins for the Bloch-periodic (k-point) oracle (oracle/bloch_oracle.py).  CPU only.

Independent ground truths: the closed-form Bloch spectrum of a circulant-with-phase stencil; the REAL oracle
(oracle/exx_oracle.py, pinned on its own) at theta = 0 and through the supercell identity; a dense complex
N x N Laplacian assembled point by point with the golden textbook weights; Hermiticity and gauge invariance.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import bloch_oracle as blo
from oracle import exx_oracle as orc

P, D = blo.PERIODIC, blo.DIRICHLET


def _weights(golden_dir, order, h):
    with open(os.path.join(golden_dir, "fd_second_derivative_weights.txt")) as f:
        for line in f:
            p = line.split()
            if p and p[0] == str(order):
                return [float(Fraction(x)) / h ** 2 for x in p[1:]]
    raise KeyError(order)


@pytest.mark.parametrize("n,theta", [(16, 0.7), (13, -2.1), (48, np.pi), (9, 0.0)])
def test_bloch_spectrum_closed_form_and_plane_waves(n, theta, golden_dir):
    h = 0.3
    w = _weights(golden_dir, 12, h)
    K = blo.bloch_second_derivative_matrix(n, h, P, 12, theta)
    assert np.allclose(K, K.conj().T)
    m = np.arange(n)
    lam = np.array([w[0] + 2 * sum(w[s] * np.cos((2 * np.pi * mm + theta) * s / n) for s in range(1, 7)) for mm in m])
    assert np.allclose(np.sort(np.linalg.eigvalsh(K)), np.sort(lam), rtol=0, atol=1e-12 * abs(w[0]))
    i = np.arange(n)
    for mm in (0, 1, n - 1):
        v = np.exp(1j * (2 * np.pi * mm + theta) * i / n)          # u(x + n h) = exp(i theta) u(x)
        assert np.allclose(K @ v, lam[mm] * v, rtol=0, atol=1e-11 * abs(w[0]))


def test_theta_zero_is_the_real_oracle():
    dims, bc, h = (7, 6, 5), (P, P, D), 0.4
    rng = np.random.default_rng(2)
    psi = rng.standard_normal((3, 5, 6, 7))
    occ = np.array([2.0, 1.0, 0.5])
    for omega in (0.0, 0.2):
        pb = blo.make_plan(*dims, h, bc, 12, omega, (0.0, 0.0, 0.0))
        pr = orc.make_plan(*dims, h, bc, 12, omega)
        vb, eb = blo.exx_apply_bloch(pb, psi, occ, psi)
        vr, er, _ = orc.exx_apply(pr, psi, occ, psi)
        assert np.abs(vb.imag).max() < 1e-13 * np.abs(vr).max()
        assert np.abs(vb.real - vr).max() < 1e-12 * np.abs(vr).max()
        assert np.allclose(eb, er, rtol=1e-12)


@pytest.mark.parametrize("M,p,omega", [(2, 1, 0.0), (3, 1, 0.106), (3, 2, 0.0)])
def test_supercell_identity_against_the_real_oracle(M, p, omega):
    """A function with Bloch phase theta = 2 pi p / M along x is periodic on M cells: the REAL periodic oracle
    on the M-fold supercell must reproduce the Bloch solve (real and imaginary parts separately)."""
    nx, ny, nz, h = 6, 5, 4, 0.45
    theta = 2 * np.pi * p / M
    rng = np.random.default_rng(4)
    u = rng.standard_normal((2, nz, ny, nx)) + 1j * rng.standard_normal((2, nz, ny, nx))
    pb = blo.make_plan(nx, ny, nz, h, (P, P, D), 12, omega, (theta, 0.0, 0.0))
    yb = blo.poisson_solve(pb, u)
    big = np.concatenate([u * np.exp(1j * theta * c) for c in range(M)], axis=3)      # extended over M cells
    pr = orc.make_plan(M * nx, ny, nz, h, (P, P, D), 12, omega)
    yr = orc.poisson_solve(pr, big.real) + 1j * orc.poisson_solve(pr, big.imag)
    assert np.abs(yr[..., :nx] - yb).max() < 1e-12 * np.abs(yb).max()
    assert np.abs(yr[..., nx:2 * nx] - yb * np.exp(1j * theta)).max() < 1e-12 * np.abs(yb).max()


def _dense_bloch_laplacian(golden_dir, dims, h, bc, theta):
    w = _weights(golden_dir, 12, h)
    nx, ny, nz = dims
    N = nx * ny * nz
    L = np.zeros((N, N), dtype=np.complex128)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                row = x + nx * (y + ny * z)
                for ax in range(3):
                    for s in range(-6, 7):
                        c = [x, y, z]
                        c[ax] += s
                        ph = 1.0
                        if bc[ax] == P:
                            wraps = c[ax] // dims[ax]
                            c[ax] -= wraps * dims[ax]
                            ph = np.exp(1j * theta[ax] * wraps)
                        elif not (0 <= c[ax] < dims[ax]):
                            continue
                        L[row, c[0] + nx * (c[1] + ny * c[2])] += w[abs(s)] * ph
    return L


@pytest.mark.parametrize("dims,bc,theta", [((6, 5, 4), (P, P, P), (0.9, -0.4, 2.0)), ((5, 4, 7), (P, D, P), (np.pi, 0.0, 0.3))])
def test_solve_matches_dense_complex_laplacian(dims, bc, theta, golden_dir):
    h = 0.4
    nx, ny, nz = dims
    L = _dense_bloch_laplacian(golden_dir, dims, h, bc, theta)
    assert np.allclose(L, L.conj().T)
    rng = np.random.default_rng(6)
    C = rng.standard_normal((2, nz, ny, nx)) + 1j * rng.standard_normal((2, nz, ny, nx))
    # unscreened: direct solve of -(1/4pi) L phi = rho (nonsingular: theta != 0)
    y = blo.poisson_solve(blo.make_plan(nx, ny, nz, h, bc, 12, 0.0, theta), C)
    for b in range(2):
        ref = np.linalg.solve(-L / (4 * np.pi), C[b].ravel())
        assert np.abs(y[b].ravel() - ref).max() < 1e-12 * np.abs(ref).max()
    # screened: dense matrix function through eigh of the assembled operator
    om = 0.3
    lam, U = np.linalg.eigh(L)
    f = -4 * np.pi * np.expm1(lam / (4 * om * om)) / (-lam)
    y = blo.poisson_solve(blo.make_plan(nx, ny, nz, h, bc, 12, om, theta), C)
    for b in range(2):
        ref = U @ (f * (U.conj().T @ C[b].ravel()))
        assert np.abs(y[b].ravel() - ref).max() < 1e-12 * np.abs(ref).max()


def test_vx_is_hermitian_and_gauge_invariant_and_accumulates():
    dims, bc, h, theta = (6, 5, 4), (P, P, D), 0.4, (1.1, -0.6, 0.0)
    plan = blo.make_plan(*dims, h, bc, 12, 0.106, theta)
    rng = np.random.default_rng(8)
    shape = (4, 5, 6)
    psi = rng.standard_normal((3,) + shape) + 1j * rng.standard_normal((3,) + shape)
    occ = np.array([2.0, 1.3, 0.2])
    ab = rng.standard_normal((2,) + shape) + 1j * rng.standard_normal((2,) + shape)
    vx, e = blo.exx_apply_bloch(plan, psi, occ, ab)
    G = plan.dV * np.array([[np.vdot(ab[i], vx[j]) for j in range(2)] for i in range(2)])
    assert abs(G[0, 1] - np.conj(G[1, 0])) < 1e-12 * np.abs(G).max()      # <a|Vx b> = conj <b|Vx a>
    assert np.all(np.real(np.diag(G)) < 0) and np.allclose(e, np.real(np.diag(G)))
    vx2, _ = blo.exx_apply_bloch(plan, psi * np.exp(0.83j), occ, ab)      # global phase of the orbitals drops out
    assert np.abs(vx2 - vx).max() < 1e-12 * np.abs(vx).max()
    vx3, _ = blo.exx_apply_bloch(plan, psi[2:], occ[2:], ab, vx0=blo.exx_apply_bloch(plan, psi[:2], occ[:2], ab)[0])
    assert np.abs(vx3 - vx).max() < 1e-13 * np.abs(vx).max()              # the sum over q / j can be split
