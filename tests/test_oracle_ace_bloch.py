"""Pins for the complex (k-point) ACE oracle (oracle/ace_bloch_oracle.py; PAPER.md:163-253 with the complex routines of
PAPER.md:218-230).  CPU only.

Independent ground truths: the defining property V~ Psi = W with W from the pinned Bloch exchange oracle (nonzero phase)
and from a synthetic Hermitian negative definite operator; the projector form W (h^3 Psi^H W)^-1 W^H h^3 through a
general dense complex solve; the real ACE oracle on purely real input; a textbook complex Cholesky written as loops; an
explicit inverse; a double loop for the Gram matrix; Hermiticity, negativity and gauge invariance of V~.
"""
import numpy as np
import pytest

from oracle import ace_bloch_oracle as acec
from oracle import ace_oracle as ace
from oracle import bloch_oracle as blo

P, D = blo.PERIODIC, blo.DIRICHLET


def _setup(dims=(7, 6, 5), bc=(P, P, D), omega=0.106, theta=(0.9, -1.7, 0.4), n=5, seed=3):
    nx, ny, nz = dims
    h = 0.45
    plan = blo.make_plan(nx, ny, nz, h, bc, 12, omega, theta)
    rng = np.random.default_rng(seed)
    psi = rng.standard_normal((n, nz, ny, nx)) + 1j * rng.standard_normal((n, nz, ny, nx))
    q, _ = np.linalg.qr(psi.reshape(n, -1).T)
    psi = (q.T / np.sqrt(plan.dV)).reshape(n, nz, ny, nx)
    occ = np.linspace(2.0, 0.3, n)
    W, _ = blo.exx_apply_bloch(plan, psi, occ, psi)
    return plan, psi, occ, W


def test_gram_matches_double_loop_and_is_hermitian_negative_definite():
    plan, psi, occ, W = _setup()
    M = acec.ace_gram_c(psi, W, plan.dV)
    n = psi.shape[0]
    for a in range(n):
        for b in range(n):
            s = 0.0 + 0.0j
            for x, y in zip(psi[a].ravel(), W[b].ravel()):
                s += (x.real - 1j * x.imag) * y
            assert abs(M[a, b] - plan.dV * s) < 1e-12 * np.abs(M).max()
    assert np.abs(M - M.conj().T).max() < 1e-13 * np.abs(M).max()     # Vx is Hermitian (Eq. 1)
    assert np.abs(M.imag).max() > 1e-3 * np.abs(M).max()               # a genuinely complex case
    assert np.linalg.eigvalsh(0.5 * (M + M.conj().T)).max() < 0        # and negative definite on span(Psi): R17


def test_cholesky_matches_textbook_complex_loops():
    plan, psi, occ, W = _setup(n=6)
    M = acec.ace_gram_c(psi, W, plan.dV)
    R = acec.ace_cholesky_c(M)
    A = -0.5 * (M + M.conj().T)
    n = A.shape[0]
    L = np.zeros_like(A)
    for j in range(n):                                                 # Cholesky-Banachiewicz, complex, written out
        for i in range(j, n):
            s = A[i, j]
            for k in range(j):
                s -= L[i, k] * np.conj(L[j, k])
            L[i, j] = np.sqrt(s.real) if i == j else s / L[j, j]
    assert np.allclose(R, L, rtol=0, atol=1e-13 * np.abs(L).max())
    assert np.allclose(np.triu(R, 1), 0.0) and np.abs(np.diag(R).imag).max() == 0.0 and np.diag(R).real.min() > 0
    assert np.allclose(R @ R.conj().T, A, rtol=0, atol=1e-14 * np.abs(A).max())


def test_not_positive_definite_is_an_error():
    with pytest.raises(np.linalg.LinAlgError):
        acec.ace_cholesky_c(np.eye(3, dtype=complex))


def test_xi_matches_explicit_inverse_and_normalisation():
    plan, psi, occ, W = _setup()
    xi, M = acec.ace_build_c(psi, W, plan.dV)
    R = acec.ace_cholesky_c(M)
    n = psi.shape[0]
    # column convention: xi = W R^-H, i.e. rows: xi = (R^-H)^T W = conj(R^-1) W
    ref = (np.conj(np.linalg.inv(R)) @ W.reshape(n, -1)).reshape(W.shape)
    assert np.allclose(xi, ref, rtol=0, atol=1e-12 * np.abs(ref).max())
    # h^3 Psi^H xi = M R^-H = -R
    S = plan.dV * psi.reshape(n, -1).conj() @ xi.reshape(n, -1).T
    assert np.allclose(S, -R, rtol=0, atol=1e-12 * np.abs(R).max())


@pytest.mark.parametrize("dims,bc,omega,theta", [((7, 6, 5), (P, P, D), 0.106, (0.9, -1.7, 0.4)),
                                                 ((6, 6, 6), (P, P, P), 0.0, (2.0, 0.0, -0.6)),
                                                 ((5, 8, 6), (D, P, D), 0.3, (0.0, np.pi, 0.0))])
def test_ace_reproduces_vx_on_its_own_orbitals(dims, bc, omega, theta):
    """V~ Psi = W: -xi xi^H Psi h^3 = -W R^-H R^-1 M^H = W."""
    plan, psi, occ, W = _setup(dims, bc, omega, theta)
    xi, _ = acec.ace_build_c(psi, W, plan.dV)
    out = acec.ace_apply_c(xi, psi, plan.dV)
    assert np.abs(out - W).max() < 1e-11 * np.abs(W).max()


def test_ace_with_a_synthetic_hermitian_negative_operator():
    """No exchange at all: W = A Psi with A = -B B^H (dense, Hermitian, negative definite); then V~ phi = A phi for every
    phi in span(Psi), and V~ Psi = W."""
    rng = np.random.default_rng(17)
    N, n, dV = 60, 4, 0.2
    B = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    A = -(B @ B.conj().T) / N
    psi = rng.standard_normal((n, N)) + 1j * rng.standard_normal((n, N))
    W = (A @ psi.T).T
    xi, M = acec.ace_build_c(psi, W, dV)
    assert np.abs(acec.ace_apply_c(xi, psi, dV) - W).max() < 1e-11 * np.abs(W).max()
    c = rng.standard_normal((2, n)) + 1j * rng.standard_normal((2, n))
    phi = c @ psi
    assert np.abs(acec.ace_apply_c(xi, phi, dV) - (A @ phi.T).T).max() < 1e-10 * np.abs(W).max()


def test_projector_form_hermiticity_negativity():
    plan, psi, occ, W = _setup()
    n = psi.shape[0]
    xi, M = acec.ace_build_c(psi, W, plan.dV)
    rng = np.random.default_rng(11)
    phi = rng.standard_normal((3,) + psi.shape[1:]) + 1j * rng.standard_normal((3,) + psi.shape[1:])
    Wm, Pm = W.reshape(n, -1), phi.reshape(3, -1)
    # V~ = W Ms^-1 W^H h^3 (columns); rows: out_c = sum_a X[a, c] W_a with Ms X = h^3 conj(W) Phi^T
    X = np.linalg.solve(0.5 * (M + M.conj().T), plan.dV * Wm.conj() @ Pm.T)
    ref = X.T @ Wm
    out = acec.ace_apply_c(xi, phi, plan.dV).reshape(3, -1)
    assert np.abs(out - ref).max() < 1e-11 * np.abs(ref).max()
    G = plan.dV * Pm.conj() @ out.T                                    # <phi_a | V~ phi_b>
    assert np.abs(G - G.conj().T).max() < 1e-12 * np.abs(G).max()
    assert np.linalg.eigvalsh(0.5 * (G + G.conj().T)).max() <= 1e-12 * np.abs(G).max()


def test_real_input_reduces_to_the_real_ace_oracle():
    rng = np.random.default_rng(2)
    N, n, dV = 50, 5, 0.3
    Bm = rng.standard_normal((N, N))
    A = -(Bm @ Bm.T) / N
    psi = rng.standard_normal((n, N))
    W = (A @ psi.T).T
    phi = rng.standard_normal((3, N))
    xi_r, M_r = ace.ace_build(psi, W, dV)
    xi_c, M_c = acec.ace_build_c(psi + 0j, W + 0j, dV)
    assert np.abs(M_c.imag).max() == 0.0 and np.allclose(M_c.real, M_r, rtol=0, atol=1e-14 * np.abs(M_r).max())
    assert np.abs(xi_c.imag).max() == 0.0 and np.allclose(xi_c.real, xi_r, rtol=0, atol=1e-12 * np.abs(xi_r).max())
    out_r, out_c = ace.ace_apply(xi_r, phi, dV), acec.ace_apply_c(xi_c, phi + 0j, dV)
    assert np.allclose(out_c.real, out_r, rtol=0, atol=1e-12 * np.abs(out_r).max()) and np.abs(out_c.imag).max() == 0.0


def test_invariant_under_a_global_phase_and_unitary_mixing_of_the_orbitals():
    """V~ depends on span(Psi) and on Vx only: Psi -> U Psi (with W -> U W, Vx being linear) leaves V~ phi unchanged;
    a global phase is the 1 x 1 case."""
    plan, psi, occ, W = _setup()
    n = psi.shape[0]
    rng = np.random.default_rng(4)
    phi = rng.standard_normal((2,) + psi.shape[1:]) + 1j * rng.standard_normal((2,) + psi.shape[1:])
    xi, _ = acec.ace_build_c(psi, W, plan.dV)
    base = acec.ace_apply_c(xi, phi, plan.dV)
    U, _ = np.linalg.qr(rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n)))
    for mix in (np.exp(0.7j) * np.eye(n), U):
        psi2 = np.tensordot(mix, psi, axes=(1, 0))
        W2 = np.tensordot(mix, W, axes=(1, 0))
        xi2, _ = acec.ace_build_c(psi2, W2, plan.dV)
        assert np.abs(acec.ace_apply_c(xi2, phi, plan.dV) - base).max() < 1e-11 * np.abs(base).max()
