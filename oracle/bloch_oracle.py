"""Plain complex FP64 CPU oracle for the Bloch-periodic (k-point) variant of the exact-exchange apply.

TEST INFRASTRUCTURE.  Slow, obvious, numpy only.  Shares no code with the CUDA path; imports nothing from
``paper_2501_16572_b200`` (and nothing from the real-valued oracle either: the tests compare the two).

What the paper says (PAPER.md:38-49, Eqs. 1-3; :159): with Brillouin-zone sampling the orbitals are complex,
    V_X phi_nk = - sum_{m q} w_q g_mq psi_mq (.) phi_{mq,nk},
    -(1/4pi) lap phi_{mq,nk} = conj(psi_mq) (.) phi_nk            (and the screened operator of Eq. 3),
"subject to Bloch boundary conditions at the wavevector k-q in the directions that the system is extended, and
Dirichlet boundary conditions in the directions of vacuum", and f(L) is evaluated with the same Kronecker
formalism with V^{*T} / V (Eqs. 6-7), now complex ("cublasZgemm").

Readings (R18-R20):
  R18  Bloch condition on a periodic axis a with n points and period n*h: u(x + n h) = exp(i theta_a) u(x),
       theta_a = (k-q)_a * n_a * h.  The 1-D FD matrix is the periodic one with every wrapped stencil entry
       multiplied by exp(i theta * wraps): K[i, (i+s) mod n] += w_|s| * exp(i theta * floor((i+s)/n)).  It is
       Hermitian; K = V diag(lam) V^H with real lam <= 0.  Dirichlet axes are unchanged (theta ignored).
  R19  One call handles ONE (k, q) pair: all psi_j share the phase theta^q, all targets share theta^k, and the
       plan is built for theta = theta^k - theta^q.  The caller sums over q (accumulate flag) and passes
       occ_j = w_q * g_jq (used verbatim, as R8).  f, the zero-mode rule (R3: only |lam_sum| below the threshold,
       which needs theta = 0 on every axis) and the grid inner product are those of the real case.
  R20  e_k = h^3 Re <tgt_k, vx_k> (the exchange energy is real; the imaginary part is rounding).

Layout: a complex grid function is ``[nz, ny, nx]`` complex128 here; the C ABI uses two real planes ``[2][N]``
(real part, imaginary part), which the tests convert.

Pins (tests/test_oracle_bloch.py): closed-form Bloch spectrum lam_m = w_0 + 2 sum_s w_s cos((2 pi m + theta) s / n)
with plane-wave eigenvectors; theta = 0 equals the real oracle; supercell identity (a Bloch function with
theta = 2 pi p / M is a periodic function on M cells: the REAL oracle on the supercell must give the same
solution); dense complex N x N Laplacian assembled point by point (solve / eigh); Hermiticity of Vx; invariance
under a global phase of the orbitals.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

PERIODIC = 0
DIRICHLET = 1
ZERO_MODE_REL_TOL = 1e-8


def fd_weights(order: int, h: float) -> np.ndarray:
    """Central second-derivative weights, order = 2*n0 (R4); same closed form as the real case."""
    n0 = order // 2
    f = math.factorial
    w = np.zeros(n0 + 1)
    for s in range(1, n0 + 1):
        w[s] = 2.0 * (-1.0) ** (s + 1) * f(n0) ** 2 / (s * s * f(n0 - s) * f(n0 + s))
    w[0] = -2.0 * np.sum(w[1:])
    return w / (h * h)


def bloch_second_derivative_matrix(n: int, h: float, bc: int, order: int, theta: float) -> np.ndarray:
    """Hermitian n x n matrix of d^2/dx^2 under u(x + n h) = exp(i theta) u(x) (R18)."""
    w = fd_weights(order, h)
    n0 = order // 2
    K = np.zeros((n, n), dtype=np.complex128)
    for i in range(n):
        for s in range(-n0, n0 + 1):
            j = i + s
            if bc == PERIODIC:
                wraps = j // n                      # floor division: -1, 0, +1, ...
                K[i, j - wraps * n] += w[abs(s)] * np.exp(1j * theta * wraps)
            elif 0 <= j < n:
                K[i, j] += w[abs(s)]
    return K


def kernel_multiplier(lam_sum: np.ndarray, omega: float, zero_tol: float) -> np.ndarray:
    """f per eigenvalue (Eq. 5 with reading R1): 4 pi/mu or 4 pi (1 - exp(-mu/4w^2))/mu, mu = -lam_sum."""
    mu = -lam_sum
    small = np.abs(lam_sum) < zero_tol
    safe = np.where(small, 1.0, mu)
    if omega > 0:
        m = -4.0 * np.pi * np.expm1(-safe / (4.0 * omega * omega)) / safe
        return np.where(small, np.pi / (omega * omega), m)
    return np.where(small, 0.0, 4.0 * np.pi / safe)


@dataclass
class BlochPlan:
    nx: int
    ny: int
    nz: int
    h: float
    bc: tuple
    theta: tuple
    lam: tuple
    V: tuple          # complex unitary, columns = eigenvectors
    mult: np.ndarray  # real [nz, ny, nx]

    @property
    def dV(self) -> float:
        return self.h ** 3


def make_plan(nx, ny, nz, h, bc, order, omega, theta) -> BlochPlan:
    lam, V = [], []
    for n, b, t in zip((nx, ny, nz), bc, theta):
        l, v = np.linalg.eigh(bloch_second_derivative_matrix(n, h, b, order, t))
        lam.append(l)
        V.append(v)
    zero_tol = ZERO_MODE_REL_TOL * 3.0 * abs(fd_weights(order, h)[0])
    lam_sum = lam[2][:, None, None] + lam[1][None, :, None] + lam[0][None, None, :]
    return BlochPlan(nx, ny, nz, float(h), tuple(bc), tuple(float(t) for t in theta), tuple(lam), tuple(V),
                     kernel_multiplier(lam_sum, omega, zero_tol))


def poisson_solve(plan: BlochPlan, C: np.ndarray) -> np.ndarray:
    """Y = f(L) C for a complex stack C[b, z, y, x]: project with V^H (Eq. 11b), multiply (Eq. 16), expand with V."""
    C = np.asarray(C, dtype=np.complex128)
    Vx, Vy, Vz = plan.V
    nb, nz, ny, nx = C.shape
    T = np.matmul(C, Vx.conj())                                   # T[..., a] = sum_x conj(Vx[x, a]) C[..., x]
    T = np.matmul(Vy.conj().T, T)
    T = np.matmul(Vz.conj().T, T.reshape(nb, nz, ny * nx))
    T = T * plan.mult.reshape(1, nz, ny * nx)
    Y = np.matmul(Vz, T).reshape(nb, nz, ny, nx)
    Y = np.matmul(Vy, Y)
    return np.matmul(Y, Vx.T)                                      # Y[..., x] = sum_a Vx[x, a] T[..., a]


def exx_apply_bloch(plan: BlochPlan, psi: np.ndarray, occ: np.ndarray, tgt: np.ndarray, vx0: np.ndarray | None = None):
    """vx_k = vx0_k - sum_j occ_j psi_j (.) f(L_theta)(conj(psi_j) (.) tgt_k), j ascending (Eqs. 1-3; R19);
    returns (vx, e_k) with e_k = h^3 Re <tgt_k, vx_k> (R20)."""
    psi = np.asarray(psi, dtype=np.complex128)
    tgt = np.asarray(tgt, dtype=np.complex128)
    vx = np.zeros_like(tgt) if vx0 is None else np.array(vx0, dtype=np.complex128)
    e_k = np.zeros(tgt.shape[0])
    for k in range(tgt.shape[0]):
        phi = poisson_solve(plan, psi.conj() * tgt[k][None])
        for j in range(psi.shape[0]):
            vx[k] -= occ[j] * psi[j] * phi[j]
        e_k[k] = plan.dV * np.real(np.vdot(tgt[k], vx[k]))
    return vx, e_k
