"""GPU parity of the Bloch-periodic (k-point) complex variant (exx_poisson_solve_bloch / exx_apply_bloch;
SURVEY.md 8(f) NEXT-3) against oracle/bloch_oracle.py, 1e-10 relative in the max norm (complex modulus)."""
import numpy as np
import pytest
import torch

from oracle import bloch_oracle as blo
from paper_2501_16572_b200 import exx

pytestmark = pytest.mark.gpu
TOL = 1e-10
# (kernel variant, form of the phase axes): the real form (butterfly + real products, the default), the embedded complex
# products (exx_plan_create_bloch_form, the cross-check form), and the plain kernels
VARIANTS = [pytest.param((exx.VARIANT_FUSED_DMMA, 0), id="fused_dmma"),
            pytest.param((exx.VARIANT_FUSED_DMMA, 1), id="fused_dmma_embedded"),
            pytest.param((exx.VARIANT_REFERENCE, 0), id="reference")]


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as ge
    ge.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"


def _planar(z):          # complex [n, nz, ny, nx] -> device [n, 2, nz, ny, nx]
    return torch.from_numpy(np.ascontiguousarray(np.stack([z.real, z.imag], axis=1))).cuda()


def _cplx(t):
    a = t.cpu().numpy()
    return a[:, 0] + 1j * a[:, 1]


def _rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def _rand(rng, n, dims):
    nx, ny, nz = dims
    return rng.standard_normal((n, nz, ny, nx)) + 1j * rng.standard_normal((n, nz, ny, nx))


# (dims, bc, theta, omega, n_rhs, n_c): all-complex, mixed real/complex axes, Dirichlet, odd nx (plain-kernel fallback)
SOLVE_CASES = [
    ((16, 16, 16), (0, 0, 0), (0.9, -0.4, 2.0), 0.0, 5, 2),
    ((16, 16, 16), (0, 0, 0), (np.pi, 0.0, 0.0), 0.106, 3, 4),
    ((20, 12, 9), (0, 1, 0), (0.5, 0.3, -1.2), 0.106, 4, 3),
    ((13, 8, 10), (0, 0, 1), (1.0, 2.0, 0.7), 0.0, 3, 2),
    ((48, 48, 48), (0, 0, 0), (np.pi / 2, 0.0, np.pi / 3), 0.106, 3, 2),
    ((60, 60, 120), (0, 0, 1), (0.8, -0.8, 0.0), 0.106, 2, 2),
    # single-launch embedded complex products on every axis, ragged last stages (n % 16 = 10, 12, 12) and column chunks
    ((26, 44, 60), (0, 0, 0), (0.7, -1.1, 0.4), 0.106, 3, 2),
    # complex axes longer than 64 points: the two-launch read-modify-write path (y), the three-launch z path
    ((16, 72, 10), (0, 0, 0), (0.3, 0.9, -0.5), 0.106, 3, 3),
    ((8, 8, 100), (0, 0, 0), (0.3, 0.9, -0.5), 0.0, 2, 2),
]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("case", SOLVE_CASES, ids=lambda c: f"{c[0][0]}x{c[0][1]}x{c[0][2]}_nrhs{c[4]}")
def test_bloch_solve_matches_oracle(case, variant):
    variant, form = variant
    dims, bc, theta, omega, n_rhs, n_c = case
    nx, ny, nz = dims
    h = 0.3
    rng = np.random.default_rng(31)
    C = _rand(rng, n_rhs, dims)
    ref = blo.poisson_solve(blo.make_plan(nx, ny, nz, h, bc, 12, omega, theta), C)
    plan = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=8, device=0, theta=theta, bloch_form=form)
    plan.set_variant(variant)
    d = _planar(C)
    keep = d.clone()
    out = plan.poisson_solve_bloch(d, n_c=n_c)
    torch.cuda.synchronize()
    assert torch.equal(d, keep)
    assert _rel(_cplx(out), ref) < TOL
    if variant == exx.VARIANT_FUSED_DMMA:         # without the fused z pass (exx_plan_set_fusion bit 0)
        plan.set_fusion(0)
        out0 = plan.poisson_solve_bloch(d, n_c=n_c)
        torch.cuda.synchronize()
        assert _rel(_cplx(out0), ref) < TOL
        plan.set_fusion(15)
    if variant == exx.VARIANT_FUSED_DMMA and nx % 2 == 0:
        assert plan.tma_launch_count > 0          # the tensor-core kernels served it
    with pytest.raises(exx.ExxError):             # real entry points refuse a complex plan
        plan.poisson_solve(d.view(-1, nz, ny, nx))
    plan.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_bloch_apply_two_q_points_matches_oracle(variant):
    """Targets at k, orbitals at two q-points: two plans (theta = theta_k - theta_q), second call accumulates."""
    variant, form = variant
    dims, bc, h, omega = (16, 12, 10), (0, 0, 1), 0.35, 0.106
    nx, ny, nz = dims
    th_k = np.array([0.6, -1.0, 0.0])
    th_q = [np.array([0.0, 0.0, 0.0]), np.array([2.0, 0.5, 0.0])]
    rng = np.random.default_rng(37)
    tgt = _rand(rng, 3, dims)
    psi = [_rand(rng, 5, dims), _rand(rng, 4, dims)]
    occ = [0.25 * np.linspace(2.0, 0.1, 5), 0.75 * np.linspace(2.0, 1e-5, 4)]      # w_q * g_jq
    vx_o = None
    for q in range(2):
        o = blo.make_plan(nx, ny, nz, h, bc, 12, omega, tuple(th_k - th_q[q]))
        vx_o, e_o = blo.exx_apply_bloch(o, psi[q], occ[q], tgt, vx0=vx_o)
    d_tgt = _planar(tgt)
    vx = None
    for q in range(2):
        plan = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=8, device=0, theta=tuple(th_k - th_q[q]), bloch_form=form)
        plan.set_variant(variant)
        vx, e_k = plan.apply_bloch(_planar(psi[q]), torch.from_numpy(occ[q]).cuda(), d_tgt, vx=vx, accumulate=q > 0,
                                   n_c=3 if q == 0 else 8)
        torch.cuda.synchronize()
        plan.close()
    assert _rel(_cplx(vx), vx_o) < TOL
    assert np.abs(e_k.cpu().numpy() - e_o).max() < TOL * np.abs(e_o).max()


@pytest.mark.parametrize("form", [0, 1], ids=["real_form", "embedded"])
@pytest.mark.parametrize("cfg,n_orb,n_c,cols", [(2, 64, 512, [0, 31, 63]), (3, 16, 256, [0, 15])],
                         ids=["cfg2_48c_64orb", "cfg3_60x60x120_16orb"])
def test_bloch_apply_at_the_benchmarked_sizes(cfg, n_orb, n_c, cols, form):
    """exx_apply_bloch on the grids its throughput is quoted on, set up exactly as `bench.py --bloch --config 2` does
    (48^3, 64 complex orbitals from workloads.make_complex_orbitals, n_c 512, phases pi/2, pi/3, pi/5 on the periodic
    axes), and on the 60x60x120 slab with 16 orbitals: the GPU applies the operator to ALL targets in its own batch
    shapes (the 16-byte butterfly kernels, orbits of up to 8 points, L2-ordered blocks); the oracle computes sampled
    target columns with the full sum over the orbitals."""
    from paper_2501_16572_b200 import workloads as wl
    w = wl.WORKLOADS[cfg]
    if n_orb != w.n_orb:
        w = wl.scaled(w, n_orb, n_orb, 0)
    theta = tuple(t if b == wl.PERIODIC else 0.0 for t, b in zip((np.pi / 2, np.pi / 3, np.pi / 5), w.bc))
    d_psi = wl.make_complex_orbitals(w, "cpu").cuda()
    occ = wl.occupations(w)
    plan = exx.Plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega, max_batch=max(128, n_c), device=0, theta=theta,
                    bloch_form=form)
    tma0 = plan.tma_launch_count
    vx, e_k = plan.apply_bloch(d_psi, torch.from_numpy(occ).cuda(), d_psi, n_c=n_c)
    torch.cuda.synchronize()
    assert plan.tma_launch_count > tma0                     # the tensor-core kernels served it
    psi = _cplx(d_psi)
    o = blo.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega, theta)
    vx_o, e_o = blo.exx_apply_bloch(o, psi, occ, psi[cols])
    assert _rel(_cplx(vx[cols]), vx_o) < TOL
    e_all = e_k.cpu().numpy()
    assert np.abs(e_all[cols] - e_o).max() < TOL * np.abs(e_o).max()
    # whole block, any size: Vx is Hermitian negative semidefinite -- M_ab = <psi_a|Vx psi_b> = conj(M_ba), e_k < 0
    z = _cplx(vx).reshape(n_orb, -1)
    M = psi.reshape(n_orb, -1).conj() @ z.T
    assert np.abs(M - M.conj().T).max() < 1e-9 * np.abs(M).max()
    assert np.all(e_all < 0)
    plan.close()


def test_bloch_theta_zero_equals_the_real_apply():
    dims, bc, h, omega = (16, 16, 16), (0, 0, 0), 0.5, 0.0
    rng = np.random.default_rng(41)
    psi = rng.standard_normal((6, 16, 16, 16))
    occ = np.linspace(2.0, 0.5, 6)
    real = exx.Plan(*dims, h, bc, 12, omega, max_batch=8, device=0)
    d_psi, d_occ = torch.from_numpy(psi).cuda(), torch.from_numpy(occ).cuda()
    vx_r, e_r, _ = real.apply(d_psi, d_occ, d_psi, d_occ, n_c=6)
    zero = exx.Plan(*dims, h, bc, 12, omega, max_batch=8, device=0, theta=(0.0, 0.0, 0.0))
    vx_b, e_b = zero.apply_bloch(_planar(psi + 0j), d_occ, _planar(psi + 0j), n_c=6)
    torch.cuda.synchronize()
    z = _cplx(vx_b)
    assert np.abs(z.imag).max() == 0.0
    assert _rel(z.real, vx_r.cpu().numpy()) < 1e-13
    assert np.allclose(e_b.cpu().numpy(), e_r.cpu().numpy(), rtol=1e-12)
    real.close()
    zero.close()


def test_bloch_empty_and_errors():
    plan = exx.Plan(8, 8, 8, 0.5, (0, 0, 0), 12, 0.106, max_batch=4, device=0, theta=(0.3, 0.0, 0.0))
    z = torch.zeros((0, 2, 8, 8, 8), dtype=torch.float64, device="cuda")
    t = torch.ones((2, 2, 8, 8, 8), dtype=torch.float64, device="cuda")
    vx, e = plan.apply_bloch(z, torch.zeros(0, dtype=torch.float64, device="cuda"), t)
    torch.cuda.synchronize()
    assert float(vx.abs().max()) == 0.0 and float(e.abs().max()) == 0.0
    with pytest.raises(exx.ExxError) as ei:
        plan.apply_bloch(t, torch.ones(2, dtype=torch.float64, device="cuda"), t, vx=t, accumulate=True)
    assert ei.value.status == 6
    plan.close()
