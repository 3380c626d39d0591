"""Plain FP64 CPU oracle for the exact-exchange apply on a real-space FD grid.

TEST INFRASTRUCTURE.  Slow, obvious, numpy only.  Shares no code with the CUDA
path; imports nothing from ``paper_2501_16572_b200``.  Every function cites the
passage of /root/reference/PAPER.md (arxiv 2501.16572) or the DESIGN.md reading
(R1..R14, = SURVEY.md section 8(c) A1..A14) it follows.

What is computed (PAPER.md:38 Eq. 1, :42 Eq. 2, :46 Eq. 3, :57-61 Eqs. 4-5, :66-70 Eqs. 6-7,
:178 Eq. 19b; E_x per BASELINE.json north_star):

    vx_k = - sum_j occ_j * psi_j (.) [ f(L) (psi_j (.) tgt_k) ]
    e_k  = h^3 * <tgt_k, vx_k>,      E_x = 1/2 * sum_k occ_tgt_k * e_k

with L = I(x)I(x)Kx + I(x)Ky(x)I + Kz(x)I(x)I (x fastest), K_a the 1-D FD matrix of
+d^2/dx^2, and f evaluated exactly through the per-axis eigendecompositions
(the method is not an approximation: the oracle IS the definition, written with
the separable evaluation of Eq. 7; tests pin it against dense N x N evaluations).

Array layout everywhere: a grid function is ``[nz, ny, nx]`` (x fastest, the paper's
vec of an n1 x n2 x n3 array with frontal slices X(:,:,k)); a set of
functions is ``[n, nz, ny, nx]`` (the column blocks of Eq. 10).

Parity pins (tests/test_oracle_*.py, ``-m "not gpu"``): FD weights (rationals, polynomial
exactness), periodic spectrum closed form, order-2 Dirichlet sine spectrum, dense direct
solve / dense matrix function of a brute-force assembled 3-D Laplacian on tiny grids,
plane-wave analytic solution, screened kernel against the numerically integrated radial
Fourier transform of erfc(w r)/r, Hermiticity / negativity / linearity / pair symmetry,
E_x double-loop identity, naive triple-loop solve, Eq. 8 per-slice solve against the batch solve.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

PERIODIC = 0
DIRICHLET = 1

ZERO_MODE_REL_TOL = 1e-8  # reading R3: |lam_sum| < 1e-8 * (|w0x|+|w0y|+|w0z|)


def fd_weights(order: int, h: float) -> np.ndarray:
    """Central FD weights w[0..n0] of the second derivative, order = 2*n0 (reading R4).

    w_q = 2 (-1)^(q+1) (n0!)^2 / (q^2 (n0-q)! (n0+q)!) / h^2 for q >= 1,
    w_0 = -2 sum_q w_q.  The "discrete Laplacian" of PAPER.md:59 with BASELINE.json's
    "FD order 12".
    """
    if order < 2 or order % 2:
        raise ValueError("order must be even and >= 2")
    if not h > 0:
        raise ValueError("h must be positive")
    n0 = order // 2
    w = np.zeros(n0 + 1, dtype=np.float64)
    f = math.factorial
    for q in range(1, n0 + 1):
        w[q] = 2.0 * (-1.0) ** (q + 1) * f(n0) ** 2 / (q * q * f(n0 - q) * f(n0 + q))
    w[0] = -2.0 * np.sum(w[1:])
    return w / (h * h)


def second_derivative_matrix(n: int, h: float, bc: int, order: int) -> np.ndarray:
    """Dense n x n matrix K of +d^2/dx^2 on one axis (readings R2, R6).

    Periodic: K[i, (i+q) mod n] += w_|q| (accumulating on wrap, so n < 2*n0+1 is defined).
    Dirichlet: K[i, i+q] = w_|q| only for 0 <= i+q < n (stencil truncated, zero outside).
    """
    w = fd_weights(order, h)
    n0 = order // 2
    K = np.zeros((n, n), dtype=np.float64)
    for i in range(n):
        for q in range(-n0, n0 + 1):
            j = i + q
            if bc == PERIODIC:
                K[i, j % n] += w[abs(q)]
            elif bc == DIRICHLET:
                if 0 <= j < n:
                    K[i, j] = w[abs(q)]
            else:
                raise ValueError("bc must be PERIODIC (0) or DIRICHLET (1)")
    return K


def kernel_multiplier(lam_sum: np.ndarray, omega: float, zero_tol: float) -> np.ndarray:
    """f(Lambda) of PAPER.md:61 (Eq. 5), per eigenvalue of L (readings R1, R2, R3).

    mu = -lam_sum >= 0.
    unscreened (omega <= 0): 4 pi / mu, and 0 where |lam_sum| < zero_tol (dropped zero mode).
    screened   (omega  > 0): 4 pi (1 - exp(-mu / (4 omega^2))) / mu, written with expm1, and
                             its limit pi / omega^2 where |lam_sum| < zero_tol.
    """
    lam_sum = np.asarray(lam_sum, dtype=np.float64)
    mu = -lam_sum
    small = np.abs(lam_sum) < zero_tol
    safe_mu = np.where(small, 1.0, mu)
    if omega > 0:
        m = -4.0 * np.pi * np.expm1(-safe_mu / (4.0 * omega * omega)) / safe_mu
        return np.where(small, np.pi / (omega * omega), m)
    m = 4.0 * np.pi / safe_mu
    return np.where(small, 0.0, m)


@dataclass
class OraclePlan:
    nx: int
    ny: int
    nz: int
    h: float
    bc: tuple
    order: int
    omega: float
    lam: tuple      # (lam_x, lam_y, lam_z), ascending as numpy.linalg.eigh returns them
    V: tuple        # (Vx, Vy, Vz), columns = eigenvectors
    mult: np.ndarray  # [nz, ny, nx] multiplier m(lam_x[a] + lam_y[b] + lam_z[c]) at [c, b, a]

    @property
    def N(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def dV(self) -> float:
        return self.h ** 3


def make_plan(nx, ny, nz, h, bc, order=12, omega=0.0) -> OraclePlan:
    """Per-axis eigendecompositions K_a = V_a diag(lam_a) V_a^T (Eqs. 6-7)
    and the multiplier table f(Lambda~) (Eq. 16)."""
    dims = (nx, ny, nz)
    lam, V = [], []
    for n, b in zip(dims, bc):
        K = second_derivative_matrix(n, h, b, order)
        l, v = np.linalg.eigh(K)
        lam.append(l)
        V.append(v)
    w0 = abs(fd_weights(order, h)[0])
    zero_tol = ZERO_MODE_REL_TOL * 3.0 * w0
    lam_sum = lam[2][:, None, None] + lam[1][None, :, None] + lam[0][None, None, :]
    mult = kernel_multiplier(lam_sum, omega, zero_tol)
    return OraclePlan(nx, ny, nz, float(h), tuple(bc), order, float(omega),
                      tuple(lam), tuple(V), mult)


def poisson_solve(plan: OraclePlan, C: np.ndarray) -> np.ndarray:
    """Y = f(L) C for a stack C[b, z, y, x] (PAPER.md:86 Eq. 9, :96-98 Eq. 11).

    Forward: project on the eigenvectors (V^T, reading R11); Hadamard with f(Lambda~)
    broadcast over the batch (Eq. 16); backward: expand with V.
    """
    C = np.asarray(C, dtype=np.float64)
    squeeze = C.ndim == 3
    if squeeze:
        C = C[None]
    Vx, Vy, Vz = plan.V
    nb, nz, ny, nx = C.shape
    # each mode product is one (broadcast) matmul -- a library primitive as a step, in Eq. 11's order
    T = np.matmul(C, Vx)                                          # T[b,z,y,a] = sum_x C[b,z,y,x] Vx[x,a]
    T = np.matmul(Vy.T, T)                                        # T[b,z,B,a] = sum_y Vy[y,B] T[b,z,y,a]
    T = np.matmul(Vz.T, T.reshape(nb, nz, ny * nx))               # T[b,c,(B,a)] = sum_z Vz[z,c] T[b,z,(B,a)]
    T = T * plan.mult.reshape(1, nz, ny * nx)                     # Hadamard with f(Lambda~), Eq. 16
    Y = np.matmul(Vz, T).reshape(nb, nz, ny, nx)                  # expand back: z, then y, then x
    Y = np.matmul(Vy, Y)
    Y = np.matmul(Y, Vx.T)
    return Y[0] if squeeze else Y


def poisson_solve_loops(plan: OraclePlan, c: np.ndarray) -> np.ndarray:
    """Same map as :func:`poisson_solve` for ONE right-hand side, as bare Python loops over
    the definition X = (V1(x)V2(x)V3) f(Lambda) (V1^T(x)V2^T(x)V3^T) B (Eq. 7).
    O(N^2); only for grids up to about 8^3 (cross-check of the vectorised version)."""
    nx, ny, nz = plan.nx, plan.ny, plan.nz
    Vx, Vy, Vz = plan.V
    t = np.zeros((nz, ny, nx))
    for c_ in range(nz):
        for b_ in range(ny):
            for a_ in range(nx):
                s = 0.0
                for z in range(nz):
                    for y in range(ny):
                        for x in range(nx):
                            s += Vz[z, c_] * Vy[y, b_] * Vx[x, a_] * c[z, y, x]
                t[c_, b_, a_] = s * plan.mult[c_, b_, a_]
    out = np.zeros((nz, ny, nx))
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                s = 0.0
                for c_ in range(nz):
                    for b_ in range(ny):
                        for a_ in range(nx):
                            s += Vz[z, c_] * Vy[y, b_] * Vx[x, a_] * t[c_, b_, a_]
                out[z, y, x] = s
    return out


def poisson_solve_eq8(plan: OraclePlan, b: np.ndarray) -> np.ndarray:
    """The NON-batch Kronecker solve of ONE right-hand side, PAPER.md:74-78 (Eq. 8a/8b), step by step in the
    paper's order: for every frontal slice B_k = B(:,:,k) (an n1 x n2 matrix, here b[k].T since arrays are
    [z, y, x]) the two small products V1^T B_k V2; the slices stacked into an (n1 n2) x n3 matrix times V3; the
    Hadamard product with f(Lambda~); then the same back: times V3^T, and V1 X~_k V2^T per slice.  That is the
    paper's 4 n3 + 2 dense products.  Pinned by equality with :func:`poisson_solve` (itself pinned to the dense
    direct solve) and with :func:`poisson_solve_loops`; the Fig. 2 comparison line of SURVEY.md 8(f) NEXT-4."""
    b = np.asarray(b, dtype=np.float64)
    V1, V2, V3 = plan.V                                      # x, y, z
    n1, n2, n3 = plan.nx, plan.ny, plan.nz
    T = np.empty((n1 * n2, n3))
    for k in range(n3):                                      # 2 n3 products
        Bk = b[k].T                                          # B(:,:,k): [x, y]
        T[:, k] = ((V1.T @ Bk) @ V2).reshape(n1 * n2, order="F")   # vec over (x fastest, then y)
    Xt = T @ V3                                              # 1 product: [(a,b), c]
    Xt = Xt * plan.mult.reshape(n3, n2 * n1).T               # f(Lambda~) (.) ..., table entry [c, b, a]
    Y = Xt @ V3.T                                            # 1 product: [(a,b), k]
    out = np.empty((n3, n2, n1))
    for k in range(n3):                                      # 2 n3 products
        Xk = Y[:, k].reshape(n1, n2, order="F")
        out[k] = ((V1 @ Xk) @ V2.T).T
    return out


def exx_accumulate(plan: OraclePlan, psi: np.ndarray, occ: np.ndarray, tgt_k: np.ndarray,
                   vx_k: np.ndarray, chunk: int = 16) -> None:
    """vx_k -= sum_j occ_j psi_j (.) f(L)(psi_j (.) tgt_k), j ascending (Eq. 1,
    :42 Eq. 2, :178 Eq. 19b; readings R8, R9: occ used verbatim, no thresholding)."""
    n_occ = psi.shape[0]
    for j0 in range(0, n_occ, chunk):
        j1 = min(n_occ, j0 + chunk)
        rho = psi[j0:j1] * tgt_k[None]            # pair densities (real: conj is a no-op)
        phi = poisson_solve(plan, rho)
        for j in range(j0, j1):
            vx_k -= occ[j] * psi[j] * phi[j - j0]


def exx_apply(plan: OraclePlan, psi: np.ndarray, occ: np.ndarray, tgt: np.ndarray,
              occ_tgt: np.ndarray | None = None, chunk: int = 16):
    """Full apply: returns (vx[n_tgt, nz, ny, nx], e_k[n_tgt], E_x).

    e_k = h^3 sum_r tgt_k(r) vx_k(r);  E_x = 1/2 sum_k occ_tgt_k e_k (reading R7;
    BASELINE.json north_star).  E_x is None when occ_tgt is None.
    """
    psi = np.asarray(psi, dtype=np.float64)
    tgt = np.asarray(tgt, dtype=np.float64)
    occ = np.asarray(occ, dtype=np.float64)
    n_tgt = tgt.shape[0]
    vx = np.zeros_like(tgt)
    e_k = np.zeros(n_tgt)
    for k in range(n_tgt):
        exx_accumulate(plan, psi, occ, tgt[k], vx[k], chunk=chunk)
        e_k[k] = plan.dV * np.sum(tgt[k] * vx[k])
    ex = None
    if occ_tgt is not None:
        ex = 0.5 * float(np.sum(np.asarray(occ_tgt, dtype=np.float64) * e_k))
    return vx, e_k, ex
