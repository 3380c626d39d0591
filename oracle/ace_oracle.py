"""Plain FP64 CPU oracle for the adaptively compressed exchange (ACE) tail and its application.

TEST INFRASTRUCTURE.  Slow, obvious, numpy/scipy only.  Shares no code with the CUDA path; imports
nothing from ``paper_2501_16572_b200``.  Follows PAPER.md:163-253 (Section III.A-B, Eqs. 17-20, 26-29)
in the paper's order and notation, with the DESIGN.md readings R15-R17:

    W   = [W^(1) ... W^(Ns)],  W^(n) = vx_n  (Eq. 19; the output of the exchange apply with targets = orbitals)
    M   = h^3 * Psi^T W                                   (Eq. 20; R15: grid inner product, weight h^3)
    Ms  = (M + M^T) / 2                                    (R16: M is symmetric up to rounding because Vx is
                                                            Hermitian; both sides factor the symmetrised matrix)
    -Ms = R R^T,  R lower triangular                      (R17: the paper says "Cholesky factor of M" and
                                                            V~ = xi xi^T (Eqs. 17, 20); M is negative definite
                                                            (Vx <= 0), so the factored matrix is -M and the
                                                            operator is V~ = -xi xi^T, as in the ACE paper it cites)
    xi  = W R^{-T}                                         (Eq. 18 / 26: cublasDtrsm with the Cholesky factor)
    chi = h^3 * xi^T Phi                                   (Eq. 28)
    V~ Phi = - xi chi                                      (Eqs. 27, 29)

Array layout: a set of n grid functions is ``[n, N]`` (each function contiguous, the paper's columns are
our rows): W, Psi, xi are [Ns, N]; Phi and V~Phi are [m, N]; chi is [Ns, m].

Pins (tests/test_oracle_ace.py, ``-m "not gpu"``): V~ Psi = W exactly (the defining property of ACE: the
compressed operator reproduces Vx on the orbitals it was built from); V~ equals the dense projector formula
W (Psi^T W h^3)^-1 W^T h^3 evaluated with a general dense solve on tiny grids (no Cholesky, no triangular
solve); V~ phi = Vx phi for phi in span(Psi), Vx from oracle/exx_oracle.py; Psi^T xi h^3 = -R; the Cholesky step
against a textbook unblocked factorisation written as loops; the triangular solve against an explicit inverse;
the Gram matrix against a double loop.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla


def ace_gram(psi: np.ndarray, w: np.ndarray, dV: float) -> np.ndarray:
    """M[a, b] = dV * sum_r psi_a(r) w_b(r)  (Eq. 20; cublasDgemm in Eq. 25)."""
    psi = np.asarray(psi, dtype=np.float64).reshape(psi.shape[0], -1)
    w = np.asarray(w, dtype=np.float64).reshape(w.shape[0], -1)
    return dV * (psi @ w.T)


def ace_cholesky(M: np.ndarray) -> np.ndarray:
    """Lower-triangular R with R R^T = -(M + M^T)/2 ("Cholesky factor"; R16, R17).
    Raises numpy.linalg.LinAlgError if -M is not positive definite."""
    Ms = 0.5 * (M + M.T)
    return np.linalg.cholesky(-Ms)


def ace_xi(w: np.ndarray, R: np.ndarray) -> np.ndarray:
    """xi = W R^{-T} (PAPER.md:169-171 Eq. 18, :226 Eq. 26: cublasDtrsm).  With functions as rows:
    xi[Ns, N] solves R xi = W (row b of W is sum_{a<=b} R[b, a] xi_a)."""
    w2 = np.asarray(w, dtype=np.float64).reshape(w.shape[0], -1)
    return sla.solve_triangular(R, w2, lower=True).reshape(w.shape)


def ace_build(psi: np.ndarray, w: np.ndarray, dV: float):
    """(xi, M): the ACE construction of PAPER.md:163-230 after W is available."""
    M = ace_gram(psi, w, dV)
    R = ace_cholesky(M)
    return ace_xi(w, R), M


def ace_apply(xi: np.ndarray, phi: np.ndarray, dV: float) -> np.ndarray:
    """V~ Phi = -xi (h^3 xi^T Phi), two steps as in PAPER.md:236-253 (Eqs. 27-29)."""
    xi2 = np.asarray(xi, dtype=np.float64).reshape(xi.shape[0], -1)
    phi2 = np.asarray(phi, dtype=np.float64).reshape(phi.shape[0], -1)
    chi = dV * (xi2 @ phi2.T)            # Eq. 28: chi[Ns, m]
    out = -(chi.T @ xi2)                 # Eq. 29: [m, N]
    return out.reshape(phi.shape)
