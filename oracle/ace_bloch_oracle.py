"""Plain complex128 CPU oracle for the ACE tail and its application with COMPLEX (k-point) orbitals.

TEST INFRASTRUCTURE.  Slow, obvious, numpy/scipy only.  Shares no code with the CUDA path; imports nothing from
``paper_2501_16572_b200`` and nothing from the other oracles.  Follows PAPER.md:163-253 (Section III.A-B, Eqs. 17-20,
26-29) in the paper's order for "complex-valued computations" (cublasZgemm, cusolver_zpotrf,
cublasZtrsm), with the DESIGN.md readings R15-R17 carried over to complex arithmetic (R21):

    M   = h^3 * Psi^H W                  (Eq. 20; the transpose of the real case becomes the conjugate transpose, as in
                                          cublasZgemm with CUBLAS_OP_C; R15: weight h^3)
    Ms  = (M + M^H) / 2                  (R16: M is Hermitian up to rounding because Vx is)
    -Ms = R R^H,  R lower triangular with a real positive diagonal          (R17: M is negative definite)
    xi  = W R^{-H}                       (Eq. 18 / 26: cublasZtrsm with the Cholesky factor)
    chi = h^3 * xi^H Phi                 (Eq. 28)
    V~ Phi = - xi chi                    (Eqs. 27, 29)

Array layout: a set of n complex grid functions is ``[n, N]`` complex128 (the paper's columns are our rows), so with
functions as rows: M[a, b] = h^3 sum_r conj(psi_a(r)) w_b(r); xi solves conj(R) xi = W (row b of W is
sum_{a <= b} conj(R[b, a]) xi_a); chi[a, c] = h^3 sum_r conj(xi_a(r)) phi_c(r); out_c = - sum_a chi[a, c] xi_a.

Pins (tests/test_oracle_ace_bloch.py, ``-m "not gpu"``): V~ Psi = W (the defining property of ACE) for W = Vx Psi from
the pinned Bloch oracle and from a synthetic Hermitian negative definite operator; the projector form
W (h^3 Psi^H W)^-1 W^H h^3 by a general dense complex solve (no Cholesky, no triangular solve); purely real input
reproduces the real ACE oracle; a textbook complex Cholesky written as loops; an explicit inverse for the triangular
solve; a double loop for the Gram matrix; Hermiticity and negative semidefiniteness of V~; invariance under a global
phase of the orbitals.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla


def _rows(a: np.ndarray) -> np.ndarray:
    a = np.asarray(a, dtype=np.complex128)
    return a.reshape(a.shape[0], -1)


def ace_gram_c(psi: np.ndarray, w: np.ndarray, dV: float) -> np.ndarray:
    """M[a, b] = dV * sum_r conj(psi_a(r)) w_b(r)  (Eq. 20; cublasZgemm)."""
    return dV * (_rows(psi).conj() @ _rows(w).T)


def ace_cholesky_c(M: np.ndarray) -> np.ndarray:
    """Lower-triangular R (real positive diagonal) with R R^H = -(M + M^H)/2 (cusolver_zpotrf; R16, R17).
    Raises numpy.linalg.LinAlgError if -M is not positive definite."""
    Ms = 0.5 * (M + M.conj().T)
    return np.linalg.cholesky(-Ms)


def ace_xi_c(w: np.ndarray, R: np.ndarray) -> np.ndarray:
    """xi = W R^{-H} (PAPER.md:169-171 Eq. 18, :226 Eq. 26: cublasZtrsm).  With functions as rows this is the
    lower-triangular system conj(R) xi = W."""
    return sla.solve_triangular(R.conj(), _rows(w), lower=True).reshape(np.shape(w))


def ace_build_c(psi: np.ndarray, w: np.ndarray, dV: float):
    """(xi, M): the ACE construction of PAPER.md:163-230 for complex orbitals, after W is available."""
    M = ace_gram_c(psi, w, dV)
    R = ace_cholesky_c(M)
    return ace_xi_c(w, R), M


def ace_apply_c(xi: np.ndarray, phi: np.ndarray, dV: float) -> np.ndarray:
    """V~ Phi = -xi (h^3 xi^H Phi), two steps as in PAPER.md:236-253 (Eqs. 27-29)."""
    xi2, phi2 = _rows(xi), _rows(phi)
    chi = dV * (xi2.conj() @ phi2.T)     # Eq. 28: chi[Ns, m]
    out = -(chi.T @ xi2)                 # Eq. 29: [m, N]
    return out.reshape(np.shape(phi))
