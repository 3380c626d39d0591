"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerance 1e-10 relative in the max norm on vx and on E_x
(BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

from oracle import exx_oracle as orc
from paper_2501_16572_b200 import exx, workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-10
VARIANTS = [pytest.param(exx.VARIANT_FUSED_DMMA, id="fused_dmma"), pytest.param(exx.VARIANT_REFERENCE, id="reference"),
            pytest.param(exx.VARIANT_CPASYNC, id="cpasync")]


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as ge
    ge.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"


def _rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def _oracle_plan(w):
    return orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)


SOLVE_CASES = [
    # (nx, ny, nz, h, bc, omega, n_rhs, n_c): ragged sizes (not multiples of 4/8), all BC mixes, tails
    (16, 16, 16, 0.5, (0, 0, 0), 0.0, 5, 2),
    (16, 16, 16, 0.5, (0, 0, 0), 0.106, 8, 8),
    (20, 12, 9, 0.3, (0, 1, 0), 0.106, 7, 3),
    (13, 17, 11, 0.4, (1, 1, 1), 0.0, 4, 4),
    (48, 48, 48, 0.25, (0, 0, 0), 0.106, 6, 4),
    (60, 60, 120, 0.25, (0, 0, 1), 0.106, 3, 2),
    (33, 8, 70, 0.25, (0, 0, 1), 0.0, 3, 1),
    (1, 1, 40, 0.25, (0, 0, 1), 0.106, 2, 2),
    (96, 96, 96, 0.2, (0, 0, 0), 0.106, 2, 2),
    (120, 120, 120, 0.2, (0, 0, 0), 0.106, 1, 1),
    # one axis longer than 128 points in each position: that axis runs on the plain kernel (per-axis fallback,
    # buffer swap, pending multiplier), the other two stay on the tensor-core path
    (130, 8, 6, 0.3, (0, 0, 0), 0.106, 3, 2),
    (8, 132, 6, 0.3, (1, 0, 1), 0.0, 3, 2),
    (6, 8, 136, 0.3, (0, 0, 1), 0.106, 3, 3),
    (6, 8, 136, 0.3, (0, 0, 0), 0.0, 2, 1),
]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("case", SOLVE_CASES, ids=lambda c: f"{c[0]}x{c[1]}x{c[2]}_nrhs{c[6]}_nc{c[7]}")
def test_poisson_solve_matches_oracle(case, variant):
    nx, ny, nz, h, bc, omega, n_rhs, n_c = case
    plan = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=8, device=0)
    plan.set_variant(variant)
    rng = np.random.default_rng(99)
    C = rng.standard_normal((n_rhs, nz, ny, nx))
    ref = orc.poisson_solve(orc.make_plan(nx, ny, nz, h, bc, 12, omega), C)
    d = torch.from_numpy(C).cuda()
    keep = d.clone()
    out = plan.poisson_solve(d, n_c=n_c)
    torch.cuda.synchronize()
    assert torch.equal(d, keep)                                  # input untouched
    assert _rel(out.cpu().numpy(), ref) < TOL
    out2 = plan.poisson_solve(d, out=d, n_c=n_c)                 # in place
    torch.cuda.synchronize()
    assert torch.equal(out2, out)
    if variant == exx.VARIANT_FUSED_DMMA and nx % 2 == 0:
        # two calls; per batch two passes through the TMA kernels for an x or y axis of at most 128 points and one
        # fused pass (forward + multiplier + backward) for such a z axis
        per_batch = 2 * (nx <= 128) + 2 * (ny <= 128) + 1 * (nz <= 128)
        assert plan.tma_launch_count == 2 * per_batch * ((n_rhs + n_c - 1) // n_c)
    else:
        assert plan.tma_launch_count == 0
    plan.close()


@pytest.mark.parametrize("dims,bc,omega", [((130, 8, 6), (0, 0, 0), 0.106), ((8, 132, 6), (0, 1, 0), 0.0),
                                           ((6, 8, 136), (0, 0, 1), 0.106)])
def test_apply_with_an_axis_longer_than_128(dims, bc, omega):
    """exx.h: an axis longer than 128 points falls back, per axis, to the plain kernel -- the only user of the second
    workspace half (canary-guarded here) and of the pending-multiplier hand-over."""
    nx, ny, nz = dims
    rng = np.random.default_rng(11)
    n = 5
    psi = rng.standard_normal((n, nz, ny, nx))
    occ = np.linspace(2.0, 0.2, n)
    plan = exx.Plan(nx, ny, nz, 0.3, bc, 12, omega, max_batch=8, device=0)
    o = orc.make_plan(nx, ny, nz, 0.3, bc, 12, omega)
    vx_o, e_o, ex_o = orc.exx_apply(o, psi, occ, psi[1:4], occ[1:4])
    d_psi, d_occ = torch.from_numpy(psi).cuda(), torch.from_numpy(occ).cuda()
    nbytes = plan.workspace_bytes(3)
    raw = torch.full((nbytes // 8 + 2 * 512,), -7.25e300, dtype=torch.float64, device="cuda")
    plan._ws = raw[512:512 + nbytes // 8].view(torch.uint8)
    vx, e_k, ex = plan.apply(d_psi, d_occ, d_psi[1:4], d_occ[1:4], n_c=3)
    torch.cuda.synchronize()
    assert _rel(vx.cpu().numpy(), vx_o) < TOL and abs(ex.item() - ex_o) < TOL * abs(ex_o)
    assert bool((raw[:512] == -7.25e300).all() and (raw[-512:] == -7.25e300).all())
    assert 0 < plan.tma_launch_count < plan.last_launch_count      # both kinds of kernels ran
    # in-place solve on the same plan: the result must come back into the caller's buffer after the swaps
    C = rng.standard_normal((2, nz, ny, nx))
    d = torch.from_numpy(C).cuda()
    plan.poisson_solve(d, out=d, n_c=2)
    torch.cuda.synchronize()
    assert _rel(d.cpu().numpy(), orc.poisson_solve(o, C)) < TOL
    assert bool((raw[:512] == -7.25e300).all() and (raw[-512:] == -7.25e300).all())
    plan.close()


def test_buffers_offset_by_8_bytes_take_the_cpasync_path():
    """TMA needs 16-byte aligned bases: with even nx but psi / vx / rhs offset by one double every product must fall
    back to the cp.async tensor-core kernels (exx_plan_tma_launch_count stays 0) and still match the oracle."""
    w = wl.scaled(wl.WORKLOADS[2], 6, 3, 1)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    plan = exx.Plan.for_workload(w, max_batch=8, device=0)
    N = w.N
    raw_psi = torch.zeros(6 * N + 1, dtype=torch.float64, device="cuda")
    d_psi = raw_psi[1:].view(6, w.nz, w.ny, w.nx)
    d_psi.copy_(psi)
    raw_vx = torch.zeros(3 * N + 1, dtype=torch.float64, device="cuda")
    d_vx = raw_vx[1:].view(3, w.nz, w.ny, w.nx)
    assert d_psi.data_ptr() % 16 == 8 and d_vx.data_ptr() % 16 == 8
    ws = torch.empty(plan.workspace_bytes(4) + 8, dtype=torch.uint8, device="cuda")
    plan._ws = ws[8:]
    vx, e_k, ex = plan.apply(d_psi, occ.cuda(), d_psi[1:4], occ_t.cuda(), vx=d_vx, n_c=4)
    torch.cuda.synchronize()
    vx_o, e_o, ex_o = orc.exx_apply(_oracle_plan(w), psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy())
    assert _rel(vx.cpu().numpy(), vx_o) < TOL and abs(ex.item() - ex_o) < TOL * abs(ex_o)
    assert plan.tma_launch_count == 0 and plan.last_launch_count > 0
    out = plan.poisson_solve(d_psi[:2], out=d_vx[:2], n_c=2)
    torch.cuda.synchronize()
    assert _rel(out.cpu().numpy(), orc.poisson_solve(_oracle_plan(w), psi[:2].numpy())) < TOL
    assert plan.tma_launch_count == 0
    plan.close()


@pytest.mark.parametrize("dims,bc,omega", [((16, 16, 16), (0, 0, 0), 0.0), ((20, 12, 9), (0, 1, 0), 0.106),
                                           ((13, 17, 11), (1, 1, 1), 0.106), ((48, 48, 48), (0, 0, 0), 0.106)])
def test_nonbatch_eq8_solver_matches_oracle(dims, bc, omega):
    """exx_poisson_solve_nonbatch (Eq. 8; the Fig. 2 comparison line) against the oracle's per-slice
    solve and against the batch solver; 4 nz + 2 launches per system."""
    nx, ny, nz = dims
    C = np.random.default_rng(21).standard_normal((3, nz, ny, nx))
    o = orc.make_plan(nx, ny, nz, 0.3, bc, 12, omega)
    ref = np.stack([orc.poisson_solve_eq8(o, C[b]) for b in range(3)])
    plan = exx.Plan(nx, ny, nz, 0.3, bc, 12, omega, max_batch=8, device=0)
    d = torch.from_numpy(C).cuda()
    out = plan.poisson_solve_nonbatch(d)
    torch.cuda.synchronize()
    assert plan.last_launch_count == 3 * (4 * nz + 2)
    assert _rel(out.cpu().numpy(), ref) < TOL
    assert _rel(out.cpu().numpy(), plan.poisson_solve(d, n_c=3).cpu().numpy()) < TOL
    plan.poisson_solve_nonbatch(d, out=d)          # in place
    torch.cuda.synchronize()
    assert torch.equal(d, out)
    plan.close()


FUSION_GRIDS = [
    # (nx, ny, nz, bc, omega): every ceil(n/8) class of the fused kernels, ragged last stages (n % 16 in 1..15), ragged
    # row tiles and column chunks, periodic and Dirichlet
    (16, 16, 16, (0, 0, 0), 0.0),
    (20, 12, 9, (0, 1, 0), 0.106),
    (26, 14, 30, (1, 0, 0), 0.106),
    (44, 6, 50, (0, 0, 1), 0.0),
    (60, 10, 60, (0, 0, 1), 0.106),
    (72, 6, 90, (0, 0, 0), 0.106),
    (100, 4, 114, (1, 1, 1), 0.106),
    (126, 4, 128, (0, 0, 0), 0.0),
    (8, 132, 6, (0, 0, 0), 0.106),      # y axis on the plain kernel, x and z fused
    # nx == 8 (mod 16): the y passes run on 8-column half-chunk tiles (k_mode_t HC), ragged and exact y extents
    (24, 20, 10, (0, 0, 0), 0.106),
    (40, 36, 6, (0, 1, 0), 0.0),
    (56, 64, 4, (1, 0, 0), 0.106),
    (120, 26, 8, (0, 0, 1), 0.106),
    # z axis on the reflection-adapted basis (k_mode_zz_sym), five row tiles per block: periodic even n (z = n/2 is its
    # own mirror image), Dirichlet odd n (the middle point is)
    (16, 4, 70, (0, 0, 0), 0.106),
    (16, 4, 77, (0, 0, 1), 0.0),
    # y axis on the reflection-adapted basis (k_mode_lf_sym / k_mode_lb_sym): 16-column chunks and half-chunks, periodic
    # and Dirichlet, with and without a symmetric z axis
    (16, 70, 4, (0, 0, 0), 0.106),
    (24, 77, 4, (0, 1, 0), 0.0),
    (40, 126, 5, (1, 0, 0), 0.106),
    (16, 120, 70, (0, 0, 1), 0.106),
    # x axis too (k_mode_xf_sym / k_mode_xacc_sym; nx a multiple of 4): exchange apply only
    (72, 4, 4, (0, 0, 0), 0.106),
    (124, 4, 4, (1, 0, 0), 0.0),
    (104, 6, 4, (0, 0, 0), 0.106),       # seven row tiles per block: the ten-warp x-forward kernel
    (128, 4, 4, (0, 0, 0), 0.0),         # eight full row tiles, no ragged stage: untrimmed image, eight warps
    (72, 70, 70, (0, 0, 0), 0.106),
    # three and four row tiles per block (axes of 34 .. 64 points), all three axes symmetric
    (40, 36, 34, (0, 1, 0), 0.106),
    (64, 50, 44, (1, 0, 0), 0.0),
]


@pytest.mark.parametrize("grid", FUSION_GRIDS, ids=lambda c: f"{c[0]}x{c[1]}x{c[2]}")
def test_fused_passes_match_oracle_and_unfused(grid):
    """exx_plan_set_fusion: k_mode_zz (z-forward + multiplier + z-backward) and k_mode_xacc (x-backward + accumulate)
    against the oracle and against the separate passes, for every mask, solver and apply, accumulate mode included."""
    nx, ny, nz, bc, omega = grid
    rng = np.random.default_rng(5)
    n_orb, n_tgt, t0 = 7, 3, 2
    psi = rng.standard_normal((n_orb, nz, ny, nx))
    occ = np.linspace(2.0, 0.1, n_orb)
    C = rng.standard_normal((5, nz, ny, nx))
    o = orc.make_plan(nx, ny, nz, 0.3, bc, 12, omega)
    phi_o = orc.poisson_solve(o, C)
    vx_o, e_o, ex_o = orc.exx_apply(o, psi, occ, psi[t0:t0 + n_tgt], occ[t0:t0 + n_tgt])
    plan = exx.Plan(nx, ny, nz, 0.3, bc, 12, omega, max_batch=32, device=0)
    d_psi, d_occ, d_C = torch.from_numpy(psi).cuda(), torch.from_numpy(occ).cuda(), torch.from_numpy(C).cuda()
    results = {}
    for mask in (0, 1, 2, 3, 6, 7, 9, 15):
        plan.set_fusion(mask)
        assert plan.fusion == mask
        dense = 4.0 * nx * ny * nz * (nx + ny + nz)
        assert plan.executed_flops_per_solve <= dense * (1 + 1e-12)
        if not (mask & 8) or not (mask & 1):
            assert plan.executed_flops_per_solve == dense        # symmetric mode needs bits 0 and 3
        for n_c in (3, 32):
            phi = plan.poisson_solve(d_C, n_c=n_c)
            assert _rel(phi.cpu().numpy(), phi_o) < TOL
            vx, e_k, ex = plan.apply(d_psi, d_occ, d_psi[t0:t0 + n_tgt], d_occ[t0:t0 + n_tgt], n_c=n_c)
            torch.cuda.synchronize()
            assert _rel(vx.cpu().numpy(), vx_o) < TOL, (mask, n_c)
            assert abs(ex.item() - ex_o) < TOL * abs(ex_o)
            results[(mask, n_c)] = vx.clone()
        # accumulate mode: two calls over a split of the orbitals give the full sum
        plan.set_accumulate(False)
        vx2, _, _ = plan.apply(d_psi[:4], d_occ[:4], d_psi[t0:t0 + n_tgt], n_c=32)
        plan.set_accumulate(True)
        plan.apply(d_psi[4:], d_occ[4:], d_psi[t0:t0 + n_tgt], vx=vx2, n_c=32)
        plan.set_accumulate(False)
        torch.cuda.synchronize()
        assert _rel(vx2.cpu().numpy(), vx_o) < TOL
    # the sum over j is ascending whatever the batch shape and the mask: rounding-level agreement between all runs that
    # contract with the same eigenbasis (bit 3 changes the basis: those agree with the others through the oracle bound)
    # (with bit 3 the x axis runs on its reflection-adapted basis only when bit 1 is on too: masks 9 and 15 differ in it)
    def basis(mask):
        return (mask & 8, mask & 2 if (mask & 8) and (mask & 1) else 0)

    for ref_mask in (1, 9, 15):
        ref = results[(ref_mask, 32)]
        for key, v in results.items():
            if basis(key[0]) == basis(ref_mask):
                assert float((v - ref).abs().max() / ref.abs().max()) < 1e-12, key
    plan.close()


APPLY_CASES = [
    # (cfg, n_orb, n_tgt, tgt_start, n_c)
    (1, 8, 8, 0, 0),        # BASELINE config 1, full: 64 pair solves
    (1, 8, 8, 0, 3),        # ragged batches
    (1, 8, 3, 5, 64),       # several targets per batch
    (2, 12, 12, 0, 5),
    (3, 10, 4, 3, 4),
    (4, 6, 2, 4, 4),
]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("case", APPLY_CASES, ids=lambda c: f"cfg{c[0]}_o{c[1]}_t{c[2]}_nc{c[4]}")
def test_apply_matches_oracle(case, variant):
    cfg, n_orb, n_tgt, t0, n_c = case
    w = wl.scaled(wl.WORKLOADS[cfg], n_orb, n_tgt, t0)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    if w.fermi:   # exercise fractional, tiny and exactly-zero occupations on the small case
        occ = occ.clone()
        occ[:] = torch.tensor(np.linspace(2.0, 0.05, n_orb))
        occ[-1] = 1e-13
        occ[1] = 0.0
        occ_t = occ[t0:t0 + n_tgt]
    plan = exx.Plan.for_workload(w, max_batch=64, device=0)
    plan.set_variant(variant)
    dpsi = psi.cuda()
    vx, e_k, ex = plan.apply(dpsi, occ.cuda(), dpsi[t0:t0 + n_tgt], occ_t.cuda(), n_c=n_c)
    torch.cuda.synchronize()
    vx_o, e_o, ex_o = orc.exx_apply(_oracle_plan(w), psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy())
    assert _rel(vx.cpu().numpy(), vx_o) < TOL
    assert np.abs(e_k.cpu().numpy() - e_o).max() / np.abs(e_o).max() < TOL
    assert abs(ex.item() - ex_o) / abs(ex_o) < TOL
    assert plan.last_launch_count > 0
    plan.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_config2_full_size(variant):
    # BASELINE config 2 as bench.py runs it (64 orbitals, 4,096 pair solves, default n_c)
    w = wl.WORKLOADS[2]
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    plan = exx.Plan.for_workload(w, device=0)
    plan.set_variant(variant)
    dpsi = psi.cuda()
    vx, e_k, ex = plan.apply(dpsi, occ.cuda(), dpsi, occ_t.cuda())
    torch.cuda.synchronize()
    vx_o, e_o, ex_o = orc.exx_apply(_oracle_plan(w), psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy())
    assert _rel(vx.cpu().numpy(), vx_o) < TOL
    assert abs(ex.item() - ex_o) / abs(ex_o) < TOL
    # properties that hold at any size: Hermiticity and negativity of M = Psi^T Vx Psi
    M = (dpsi.view(64, -1) @ vx.view(64, -1).T).cpu().numpy()
    assert np.abs(M - M.T).max() < 1e-10 * np.abs(M).max()
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).max() < 1e-9 * np.abs(M).max()
    plan.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_batch_size_invariance_and_determinism(variant):
    # same linear map for every n_c; only the j-summation grouping changes (rounding)
    w = wl.scaled(wl.WORKLOADS[2], 9, 4, 2)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cuda")
    plan = exx.Plan.for_workload(w, max_batch=64, device=0)
    plan.set_variant(variant)
    base, _, ex0 = plan.apply(psi, occ, tgt, occ_t, n_c=1)
    base = base.clone()
    for n_c in (2, 4, 9, 18, 64):
        v, _, ex = plan.apply(psi, occ, tgt, occ_t, n_c=n_c)
        assert float((v - base).abs().max() / base.abs().max()) < 1e-12
        assert abs(ex.item() - ex0.item()) < 1e-12 * abs(ex0.item())
    a, _, _ = plan.apply(psi, occ, tgt, occ_t, n_c=4)
    a = a.clone()
    b, _, _ = plan.apply(psi, occ, tgt, occ_t, n_c=4)
    assert torch.equal(a, b)                                  # bitwise reproducible run to run
    plan.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_edge_cases_and_errors(variant):
    w = wl.scaled(wl.WORKLOADS[1], 4, 2, 0)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cuda")
    plan = exx.Plan.for_workload(w, max_batch=8, device=0)
    plan.set_variant(variant)
    # no occupied orbitals: vx = 0, E_x = 0
    vx, e_k, ex = plan.apply(psi[:0], occ[:0], tgt, occ_t)
    torch.cuda.synchronize()
    assert float(vx.abs().max()) == 0.0 and ex.item() == 0.0 and float(e_k.abs().max()) == 0.0
    # no targets
    vx, e_k, ex = plan.apply(psi, occ, tgt[:0], occ_t[:0])
    torch.cuda.synchronize()
    assert vx.shape[0] == 0 and ex.item() == 0.0
    # all occupations zero
    vx, _, ex = plan.apply(psi, torch.zeros_like(occ), tgt, occ_t)
    torch.cuda.synchronize()
    assert float(vx.abs().max()) == 0.0
    # errors: n_c beyond max_batch, aliasing vx with psi, short workspace
    with pytest.raises((exx.ExxError, ValueError)):
        plan.apply(psi, occ, tgt, occ_t, n_c=9)
    with pytest.raises(exx.ExxError) as ei:
        plan.apply(psi, occ, tgt, occ_t, vx=psi[:2])
    assert ei.value.status == 6
    import ctypes as C
    lib = exx.load_library()
    vx = torch.empty_like(tgt)
    st = lib.exx_apply(plan._h, psi.data_ptr(), occ.data_ptr(), 4, tgt.data_ptr(), None, 2, vx.data_ptr(), None, None,
                       4, C.c_void_p(plan._workspace(8).data_ptr()), 16, None)
    assert st == 5
    plan.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_apply_host_end_to_end(variant):
    w = wl.scaled(wl.WORKLOADS[2], 6, 3, 2)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    plan = exx.Plan.for_workload(w, max_batch=16, device=0)
    plan.set_variant(variant)
    vx_h, e_h, ex_h = plan.apply_host(psi.numpy(), occ.numpy(), tgt_start=2, n_tgt=3, occ_tgt=occ_t.numpy(), n_c=4)
    vx_o, e_o, ex_o = orc.exx_apply(_oracle_plan(w), psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy())
    assert _rel(vx_h, vx_o) < TOL and abs(ex_h - ex_o) < TOL * abs(ex_o)
    # separate target block
    vx_h2, _, _ = plan.apply_host(psi.numpy(), occ.numpy(), tgt=np.ascontiguousarray(tgt.numpy()), occ_tgt=occ_t.numpy())
    assert _rel(vx_h2, vx_o) < TOL
    plan.close()


@pytest.mark.parametrize("n_orb,n_c", [(11, 4), (11, 16), (3, 2), (1, 1)])
def test_apply_host_streams_the_orbitals_in_blocks(n_orb, n_c):
    """exx_apply_host uploads the orbitals block by block (two resident) and accumulates block after block: more
    orbitals than a batch (blocks of n_c, ragged last block), fewer (four blocks), and the plan's own accumulate mode
    must not leak into the call.  Bitwise equal to the device-buffer exx_apply (same order of the sum over j)."""
    w = wl.scaled(wl.WORKLOADS[1], n_orb, min(n_orb, 5), 0)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    occ = torch.linspace(2.0, 0.3, n_orb, dtype=torch.float64)
    occ_t = occ[:w.n_tgt]
    plan = exx.Plan.for_workload(w, max_batch=16, device=0)
    vx_o, e_o, ex_o = orc.exx_apply(_oracle_plan(w), psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy())
    plan.set_accumulate(True)          # must be ignored by the host call and restored afterwards
    for _ in range(2):                 # second call reuses the plan-owned buffers (stale vx inside)
        vx_h, e_h, ex_h = plan.apply_host(psi.numpy(), occ.numpy(), tgt_start=0, n_tgt=w.n_tgt, occ_tgt=occ_t.numpy(), n_c=n_c)
        assert _rel(vx_h, vx_o) < TOL and abs(ex_h - ex_o) < TOL * abs(ex_o)
        assert np.abs(e_h - e_o).max() < TOL * np.abs(e_o).max()
    plan.set_accumulate(False)
    d_psi = psi.cuda()
    vx_d, _, _ = plan.apply(d_psi, occ.cuda(), d_psi[:w.n_tgt], occ_t.cuda(), n_c=n_c)
    torch.cuda.synchronize()
    assert np.array_equal(vx_d.cpu().numpy(), vx_h)
    plan.close()


def test_fast_variant_agrees_with_reference_variant_bitwise_close():
    w = wl.scaled(wl.WORKLOADS[3], 8, 3, 1)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cuda")
    plan = exx.Plan.for_workload(w, max_batch=16, device=0)
    out = {}
    for v in (exx.VARIANT_REFERENCE, exx.VARIANT_FUSED_DMMA):
        plan.set_variant(v)
        vx, _, ex = plan.apply(psi, occ, tgt, occ_t, n_c=8)
        out[v] = (vx.clone(), ex.item())
    a, b = out[exx.VARIANT_REFERENCE], out[exx.VARIANT_FUSED_DMMA]
    assert float((a[0] - b[0]).abs().max() / a[0].abs().max()) < 1e-12
    assert abs(a[1] - b[1]) < 1e-12 * abs(a[1])
    plan.close()


@pytest.mark.parametrize("cfg,n_orb,n_tgt,n_c", [(2, 12, 6, 4), (3, 6, 5, 3), (1, 8, 8, 8)])
def test_two_lanes_bitwise_equal_to_one_lane(cfg, n_orb, n_tgt, n_c):
    # include/exx.h exx_plan_set_lanes: target blocks alternate between two streams; every vx_k is still
    # accumulated in ascending j by one lane only, so the result must not change by a single bit
    w = wl.scaled(wl.WORKLOADS[cfg], n_orb, n_tgt, 0)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cuda")
    plan = exx.Plan.for_workload(w, max_batch=16, device=0)
    assert plan.lanes == 1
    v1, e1, x1 = plan.apply(psi, occ, tgt, occ_t, n_c=n_c)
    v1, e1, x1 = v1.clone(), e1.clone(), x1.clone()
    plan.set_lanes(2)
    assert plan.lanes == 2
    for _ in range(3):
        v2, e2, x2 = plan.apply(psi, occ, tgt, occ_t, n_c=n_c)
        torch.cuda.synchronize()
        assert torch.equal(v1, v2) and torch.equal(e1, e2) and torch.equal(x1, x2)
    o = _oracle_plan(w)
    vo, eo, xo = orc.exx_apply(o, psi.cpu().numpy(), occ.cpu().numpy(), tgt.cpu().numpy(), occ_t.cpu().numpy())
    assert _rel(v2.cpu().numpy(), vo) < TOL and abs(x2.item() - xo) < TOL * abs(xo)
    with pytest.raises(exx.ExxError):
        plan.set_lanes(3)
    plan.close()


def test_apply_is_cuda_graph_capturable():
    """include/exx.h: "The calls are CUDA-graph capturable" -- capture one exx_apply (PDL launches included) on a
    side stream, replay it twice, and compare bitwise with the eager result."""
    w = wl.scaled(wl.WORKLOADS[1], 8)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    plan = exx.Plan.for_workload(w, device=0)
    d_psi, d_occ = psi.cuda(), occ.cuda()
    vx_eager, ek_eager, ex_eager = plan.apply(d_psi, d_occ, d_psi, d_occ, n_c=4)   # also warms up attributes / tensor maps
    torch.cuda.synchronize()
    vx = torch.zeros_like(vx_eager)
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.graph(g, stream=s):
        _, ek, ex = plan.apply(d_psi, d_occ, d_psi, d_occ, vx=vx, n_c=4, stream=torch.cuda.current_stream())
    for _ in range(2):
        vx.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(vx, vx_eager) and torch.equal(ek, ek_eager) and torch.equal(ex, ex_eager)
    plan.close()


def test_accumulate_mode_splits_the_orbital_sum():
    """exx_plan_set_accumulate: the sum over occupied orbitals (Eq. 1) split over two calls -- what one rank does in
    the orbital ring (sharding.ring_apply) -- equals the oracle and the one-shot apply."""
    from paper_2501_16572_b200 import sharding
    w = wl.scaled(wl.WORKLOADS[1], 8)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    occ = torch.linspace(2.0, 0.1, 8, dtype=torch.float64)
    vx_o, e_o, ex_o = orc.exx_apply(_oracle_plan(w), psi.numpy(), occ.numpy(), tgt.numpy(), occ.numpy())
    plan = exx.Plan.for_workload(w, device=0)
    d_psi, d_occ = psi.cuda(), occ.cuda()
    vx_full, _, _ = plan.apply(d_psi, d_occ, d_psi, d_occ, n_c=4)
    vx = torch.full_like(vx_full, 7.0)                      # garbage: the first call must overwrite it
    out = {}

    def apply_block(p, o, accumulate, last):
        plan.set_accumulate(accumulate)
        out["r"] = plan.apply(p, o, d_psi, d_occ if last else None, vx=vx, n_c=4, want_ex_k=last)
        plan.set_accumulate(False)

    apply_block(d_psi[:5].contiguous(), d_occ[:5].contiguous(), False, False)
    apply_block(d_psi[5:].contiguous(), d_occ[5:].contiguous(), True, True)
    torch.cuda.synchronize()
    _, e_k, ex = out["r"]
    assert _rel(vx.cpu().numpy(), vx_o) < TOL
    assert _rel(vx.cpu().numpy(), vx_full.cpu().numpy()) < 1e-13
    assert abs(ex.item() - ex_o) < TOL * abs(ex_o)
    # the ring driver with one rank is a single plain call
    vx2 = torch.empty_like(vx)
    sharding.ring_apply(lambda p, o, accumulate, last: plan.apply(p, o, d_psi, d_occ, vx=vx2, n_c=4), d_psi, d_occ, 0, 1)
    torch.cuda.synchronize()
    assert torch.equal(vx2, vx_full)
    plan.close()


@pytest.mark.parametrize("dims,sym", [((48, 48, 48), True), ((16, 16, 16), False)], ids=["symmetric_mode", "dense"])
def test_per_pass_profile_accounts_for_every_mode_product_launch(dims, sym):
    """exx_plan_get_profile_passes (bench.py's per-kernel roofline): the passes add up to the mode-product class in
    launches and time, and their executed operations to exx_plan_executed_flops_per_solve."""
    nx, ny, nz = dims
    plan = exx.Plan(nx, ny, nz, 0.25, (0, 0, 0), 12, 0.106, max_batch=64, device=0)
    rng = np.random.default_rng(3)
    psi = torch.from_numpy(rng.standard_normal((6, nz, ny, nx))).cuda()
    occ = torch.full((6,), 2.0, dtype=torch.float64, device="cuda")
    plan.apply(psi, occ, psi, occ, n_c=12)
    plan.set_profiling(True)
    plan.apply(psi, occ, psi, occ, n_c=12)
    prof = plan.get_profile()
    passes = plan.get_profile_passes()
    plan.set_profiling(False)
    assert set(passes) == {"x_forward", "y_forward", "z", "y_backward", "x_backward"}      # fused z pass, fused accumulate
    assert sum(c for _, c, _ in passes.values()) == prof["mode_product"][1] == 5 * 3        # 36 pairs in batches of 12
    assert abs(sum(ms for ms, _, _ in passes.values()) - prof["mode_product"][0]) < 1e-6 * prof["mode_product"][0] + 1e-9
    flops = sum(f for _, _, f in passes.values())
    assert abs(flops - plan.executed_flops_per_solve) < 1e-9 * flops
    dense = 4.0 * nx * ny * nz * (nx + ny + nz)
    assert (flops < 0.6 * dense) if sym else (flops == dense)
    # one executed solve of the pair-symmetric apply runs the x-backward product once more (two-sided accumulate)
    extra = plan.executed_flops_per_symmetric_solve - plan.executed_flops_per_solve
    assert abs(extra - passes["x_backward"][2]) < 1e-9 * flops if sym else extra == 0.0
    plan.close()
