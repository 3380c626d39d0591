"""GPU parity of the ACE tail and application for COMPLEX (k-point) orbitals (exx_ace_build_bloch / exx_ace_apply_bloch;
PAPER.md:218-230, Eqs. 17-20 and 26-29 in complex arithmetic) against oracle/ace_bloch_oracle.py, element by element on
the same seeded inputs.  Tolerance as for the real ACE: M, xi and V~ Phi to 1e-10 relative in the
max norm.  W on the GPU side is the GPU's own Bloch exchange apply where a phase is given (the whole chain), or a
synthetic Hermitian negative definite operator applied on the host (the ACE steps alone, larger n)."""
import numpy as np
import pytest
import torch

from oracle import ace_bloch_oracle as acec
from oracle import bloch_oracle as blo
from paper_2501_16572_b200 import exx

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as ge
    ge.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"


def _rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def _planes(z):
    """complex [n, nz, ny, nx] -> float64 [n, 2, nz, ny, nx] (real plane, imaginary plane)."""
    return torch.from_numpy(np.ascontiguousarray(np.stack([z.real, z.imag], axis=1)))


def _cplx(t):
    a = t.cpu().numpy()
    return a[:, 0] + 1j * a[:, 1]


def _orbitals(dims, h, n, seed):
    nx, ny, nz = dims
    rng = np.random.default_rng(seed)
    psi = rng.standard_normal((n, nz, ny, nx)) + 1j * rng.standard_normal((n, nz, ny, nx))
    q, _ = np.linalg.qr(psi.reshape(n, -1).T)
    return np.ascontiguousarray((q.T / np.sqrt(h ** 3)).reshape(n, nz, ny, nx))


# (dims, bc, omega, h, theta, n_orb, n_trial): the whole chain, W from the Bloch exchange apply of each side
CHAIN = [
    ((16, 16, 16), (0, 0, 0), 0.106, 0.5, (0.9, -1.7, 0.4), 6, 4),
    ((20, 12, 9), (0, 1, 0), 0.106, 0.3, (2.0, 0.0, -0.6), 5, 3),
    ((13, 17, 11), (0, 0, 1), 0.0, 0.4, (np.pi, 0.3, 0.0), 7, 2),      # N odd: 8-byte copy path
]


@pytest.mark.parametrize("case", CHAIN, ids=lambda c: f"{c[0][0]}x{c[0][1]}x{c[0][2]}_n{c[5]}_m{c[6]}")
def test_complex_ace_after_the_bloch_exchange_apply(case):
    dims, bc, omega, h, theta, n, m = case
    nx, ny, nz = dims
    psi = _orbitals(dims, h, n, seed=17)
    occ = np.linspace(2.0, 0.05, n)
    o = blo.make_plan(nx, ny, nz, h, bc, 12, omega, theta)
    W_o, _ = blo.exx_apply_bloch(o, psi, occ, psi)
    xi_o, M_o = acec.ace_build_c(psi, W_o, o.dV)
    rng = np.random.default_rng(5)
    phi = rng.standard_normal((m, nz, ny, nx)) + 1j * rng.standard_normal((m, nz, ny, nx))
    out_o = acec.ace_apply_c(xi_o, phi, o.dV)

    plan = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=16, device=0, theta=theta)
    d_psi, d_occ = _planes(psi).cuda(), torch.from_numpy(occ).cuda()
    W, _ = plan.apply_bloch(d_psi, d_occ, d_psi, n_c=8)
    xi, M, info = plan.ace_build_bloch(d_psi, W)
    out = plan.ace_apply_bloch(xi, _planes(phi).cuda())
    torch.cuda.synchronize()
    assert int(info.item()) == 0
    Mc = M.cpu().numpy()
    assert _rel(Mc[..., 0] + 1j * Mc[..., 1], M_o) < TOL
    assert _rel(_cplx(xi), xi_o) < TOL
    assert _rel(_cplx(out), out_o) < TOL
    # the defining property on the GPU's own numbers: V~ Psi = W
    back = plan.ace_apply_bloch(xi, d_psi)
    torch.cuda.synchronize()
    assert _rel(_cplx(back), _cplx(W)) < TOL
    plan.close()


# (N as dims, n_orb, n_trial): the ACE steps alone on a synthetic Hermitian negative definite operator; several Cholesky
# blocks of 32, n not a multiple of 32, in-place xi
SYNTH = [((12, 10, 8), 5, 3), ((16, 12, 10), 40, 7), ((14, 12, 10), 97, 33), ((9, 7, 5), 64, 1)]


@pytest.mark.parametrize("case", SYNTH, ids=lambda c: f"{c[0][0]}x{c[0][1]}x{c[0][2]}_n{c[1]}_m{c[2]}")
def test_complex_ace_on_a_synthetic_operator(case):
    dims, n, m = case
    nx, ny, nz = dims
    N, h = nx * ny * nz, 0.4
    rng = np.random.default_rng(23)
    psi = _orbitals(dims, h, n, seed=3)
    B = (rng.standard_normal((N, 2 * n)) + 1j * rng.standard_normal((N, 2 * n))) / np.sqrt(N)
    W = -((psi.reshape(n, N) @ B.conj()) @ B.T).reshape(psi.shape)      # rows of (A Psi^T)^T with A = -B B^H
    W = W + 0.05 * (-(psi * 1.0))                                        # well conditioned: A - 0.05 I
    phi = rng.standard_normal((m, nz, ny, nx)) + 1j * rng.standard_normal((m, nz, ny, nx))
    dV = h ** 3
    xi_o, M_o = acec.ace_build_c(psi, W, dV)
    out_o = acec.ace_apply_c(xi_o, phi, dV)
    print("cond(-M) =", np.linalg.cond(0.5 * (M_o + M_o.conj().T)))

    plan = exx.Plan(nx, ny, nz, h, (0, 0, 0), 12, 0.106, max_batch=4, device=0)     # any plan of the grid serves
    d_psi, d_w = _planes(psi).cuda(), _planes(W).cuda()
    xi, M, info = plan.ace_build_bloch(d_psi, d_w, xi=d_w)                          # in place over W
    out = plan.ace_apply_bloch(xi, _planes(phi).cuda())
    torch.cuda.synchronize()
    assert int(info.item()) == 0 and xi.data_ptr() == d_w.data_ptr()
    Mc = M.cpu().numpy()
    assert _rel(Mc[..., 0] + 1j * Mc[..., 1], M_o) < TOL
    assert _rel(_cplx(xi), xi_o) < TOL
    assert _rel(_cplx(out), out_o) < TOL
    plan.close()


def test_complex_ace_reports_a_non_positive_pivot_and_validates():
    nx = ny = nz = 8
    plan = exx.Plan(nx, ny, nz, 0.5, (0, 0, 0), 12, 0.106, max_batch=4, device=0)
    psi = _orbitals((8, 8, 8), 0.5, 3, seed=1)
    d_psi = _planes(psi).cuda()
    _, _, info = plan.ace_build_bloch(d_psi, d_psi.clone())       # W = +Psi: M = +I, -M is not positive definite
    torch.cuda.synchronize()
    assert int(info.item()) == 1
    with pytest.raises(exx.ExxError) as ei:                        # xi overlapping psi
        plan.ace_build_bloch(d_psi, d_psi.clone(), xi=d_psi)
    assert ei.value.status == 6
    plan.close()
