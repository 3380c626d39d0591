"""Pins for the ACE oracle (oracle/ace_oracle.py; Eqs. 17-20, 26-29).  CPU only.

None of them re-types the oracle's own formula with the same routine: the defining property of ACE (the
compressed operator reproduces Vx on the orbitals it was built from, and on their span), the projector form
W M^-1 W^T evaluated with a general dense solve (no Cholesky, no triangular solve), a textbook unblocked
Cholesky written out as loops, an explicit matrix inverse for the triangular solve, a double loop for the
Gram matrix.
"""
import numpy as np
import pytest

from oracle import ace_oracle as ace
from oracle import exx_oracle as orc

P, D = orc.PERIODIC, orc.DIRICHLET


def _setup(dims=(7, 6, 5), bc=(P, P, D), omega=0.106, n=5, seed=3, occ=None):
    nx, ny, nz = dims
    h = 0.45
    plan = orc.make_plan(nx, ny, nz, h, bc, 12, omega)
    rng = np.random.default_rng(seed)
    psi = rng.standard_normal((n, nz, ny, nx))
    q, _ = np.linalg.qr(psi.reshape(n, -1).T)
    psi = (q.T / np.sqrt(plan.dV)).reshape(n, nz, ny, nx)
    occ = np.linspace(2.0, 0.3, n) if occ is None else occ
    W, _, _ = orc.exx_apply(plan, psi, occ, psi, occ)
    return plan, psi, occ, W


def test_gram_matches_double_loop_and_is_symmetric_negative_definite():
    plan, psi, occ, W = _setup()
    M = ace.ace_gram(psi, W, plan.dV)
    n = psi.shape[0]
    for a in range(n):
        for b in range(n):
            s = 0.0
            for x, y in zip(psi[a].ravel(), W[b].ravel()):
                s += x * y
            assert abs(M[a, b] - plan.dV * s) < 1e-12 * np.abs(M).max()
    assert np.abs(M - M.T).max() < 1e-13 * np.abs(M).max()      # Hermiticity of Vx (Eq. 1)
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).max() < 0         # Vx is negative definite on span(Psi): R17


def test_cholesky_matches_textbook_unblocked_loops():
    plan, psi, occ, W = _setup(n=6)
    M = ace.ace_gram(psi, W, plan.dV)
    R = ace.ace_cholesky(M)
    A = -0.5 * (M + M.T)
    n = A.shape[0]
    L = np.zeros_like(A)
    for j in range(n):                                          # Cholesky-Banachiewicz, written out
        for i in range(j, n):
            s = A[i, j]
            for k in range(j):
                s -= L[i, k] * L[j, k]
            L[i, j] = np.sqrt(s) if i == j else s / L[j, j]
    assert np.allclose(R, L, rtol=0, atol=1e-13 * np.abs(L).max())
    assert np.allclose(np.triu(R, 1), 0.0)
    assert np.allclose(R @ R.T, A, rtol=0, atol=1e-14 * np.abs(A).max())


def test_not_positive_definite_is_an_error():
    with pytest.raises(np.linalg.LinAlgError):
        ace.ace_cholesky(np.eye(3))                             # -I is not positive definite


def test_xi_matches_explicit_inverse_and_normalisation():
    plan, psi, occ, W = _setup()
    xi, M = ace.ace_build(psi, W, plan.dV)
    R = ace.ace_cholesky(M)
    n = psi.shape[0]
    ref = (np.linalg.inv(R) @ W.reshape(n, -1)).reshape(W.shape)
    assert np.allclose(xi, ref, rtol=0, atol=1e-12 * np.abs(ref).max())
    # Psi^T xi h^3 = M R^-T = -R: the overlap of the orbitals with xi is the (negated) Cholesky factor
    S = plan.dV * psi.reshape(n, -1) @ xi.reshape(n, -1).T
    assert np.allclose(S, -R, rtol=0, atol=1e-12 * np.abs(R).max())


@pytest.mark.parametrize("dims,bc,omega", [((7, 6, 5), (P, P, D), 0.106), ((6, 6, 6), (P, P, P), 0.0),
                                           ((5, 8, 6), (D, D, D), 0.3)])
def test_ace_reproduces_vx_on_its_own_orbitals(dims, bc, omega):
    """V~ Psi = W: the defining property (-xi xi^T Psi h^3 = W R^-T R^-1 M^T ... = W)."""
    plan, psi, occ, W = _setup(dims, bc, omega)
    xi, _ = ace.ace_build(psi, W, plan.dV)
    out = ace.ace_apply(xi, psi, plan.dV)
    assert np.abs(out - W).max() < 1e-11 * np.abs(W).max()


def test_ace_equals_vx_on_the_span_and_projector_form_elsewhere():
    plan, psi, occ, W = _setup()
    n = psi.shape[0]
    xi, M = ace.ace_build(psi, W, plan.dV)
    rng = np.random.default_rng(11)
    # (i) a trial function inside span(Psi): V~ phi = Vx phi (exchange apply of the oracle, linear in the target)
    c = rng.standard_normal((2, n))
    phi_in = np.tensordot(c, psi, axes=(1, 0))
    vx_in, _, _ = orc.exx_apply(plan, psi, occ, phi_in)
    assert np.abs(ace.ace_apply(xi, phi_in, plan.dV) - vx_in).max() < 1e-11 * np.abs(vx_in).max()
    # (ii) arbitrary trial functions: V~ = W M^-1 W^T h^3 with a general dense solve (no Cholesky / trsm)
    phi = rng.standard_normal((3,) + psi.shape[1:])
    Wm = W.reshape(n, -1)
    ref = (np.linalg.solve(0.5 * (M + M.T), plan.dV * Wm @ phi.reshape(3, -1).T)).T @ Wm
    out = ace.ace_apply(xi, phi, plan.dV).reshape(3, -1)
    assert np.abs(out - ref).max() < 1e-11 * np.abs(ref).max()
    # (iii) V~ is symmetric and negative semidefinite
    G = plan.dV * phi.reshape(3, -1) @ out.T
    assert np.abs(G - G.T).max() < 1e-12 * np.abs(G).max()
    assert np.linalg.eigvalsh(0.5 * (G + G.T)).max() <= 1e-12 * np.abs(G).max()


def test_ace_kills_functions_orthogonal_to_w():
    plan, psi, occ, W = _setup()
    n = psi.shape[0]
    xi, _ = ace.ace_build(psi, W, plan.dV)
    rng = np.random.default_rng(5)
    phi = rng.standard_normal((1, W[0].size))
    Wm = W.reshape(n, -1)
    coef, *_ = np.linalg.lstsq(Wm.T, phi[0], rcond=None)
    phi_perp = (phi[0] - Wm.T @ coef).reshape((1,) + psi.shape[1:])   # orthogonal to every W^(n)
    out = ace.ace_apply(xi, phi_perp, plan.dV)
    assert np.abs(out).max() < 1e-10 * np.abs(xi).max() * np.abs(phi_perp).max()
