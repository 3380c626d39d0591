"""GPU parity of the pair-symmetric exchange apply (exx_apply_symmetric) against the
oracle's full double sum (oracle/exx_oracle.exx_apply solves EVERY (j,k) pair), 1e-10 relative in the max norm
on vx and on E_x, plus the executed-solve count."""
import numpy as np
import pytest
import torch

from oracle import exx_oracle as orc
from paper_2501_16572_b200 import exx, workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as ge
    ge.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"


def _rel(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def _expected_solves(n, n_c, nk_min=1):
    """The batching rule of exx_apply_symmetric, restated: blocks of nk consecutive targets against the orbitals
    0 .. k0+nk-1 (cut into j-chunks when that exceeds n_c), nk as large as n_c allows but at least nk_min."""
    k0, total = 0, 0
    while k0 < n:
        nk = 1
        while k0 + nk + 1 <= n and (nk + 1) * (k0 + nk + 1) <= n_c:
            nk += 1
        nk = min(max(nk, nk_min), n - k0, n_c)
        total += nk * (k0 + nk)
        k0 += nk
    return total


def _nk_min(nx, ny, nz):
    """Targets per block the two-sided fused accumulate asks for (exx_api.cu): enough (at most 8) to give each of the 12
    warps of every SM a work item of 16 (up to 64 half-range x points) or 8 rows."""
    nh = (nx + 1) // 2
    rows = 16 if (nh + 7) // 8 <= 4 else 8
    tiles = (ny * nz + rows - 1) // rows
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    return max(1, min(8, (12 * sms + tiles - 1) // tiles))


# (dims, bc, omega, h, n_orb, n_c)
CASES = [
    ((16, 16, 16), (0, 0, 0), 0.0, 0.5, 8, 8),
    ((16, 16, 16), (0, 0, 0), 0.106, 0.5, 8, 1),        # every batch a single pair
    ((20, 12, 9), (0, 1, 0), 0.106, 0.3, 7, 5),         # targets with more partners than n_c: j-chunks
    ((13, 17, 11), (1, 1, 1), 0.0, 0.4, 9, 64),         # odd N, whole triangle in few rectangles
    ((24, 20, 16), (0, 0, 1), 0.106, 0.3, 37, 16),
    # every axis on the reflection-adapted basis: both sides of the accumulate fused with the x-backward product
    ((40, 36, 34), (0, 0, 1), 0.106, 0.3, 21, 16),      # j-chunks that straddle the diagonal
    ((36, 40, 44), (1, 0, 0), 0.0, 0.3, 19, 64),
    ((48, 34, 38), (0, 1, 0), 0.106, 0.25, 9, 1),       # single-pair batches
    ((72, 36, 34), (0, 0, 0), 0.106, 0.3, 12, 40),      # 8-row work items (more than 32 half-range x points)
]


@pytest.mark.parametrize("variant", [exx.VARIANT_FUSED_DMMA, exx.VARIANT_REFERENCE], ids=["fused_dmma", "reference"])
@pytest.mark.parametrize("case", CASES, ids=lambda c: f"{c[0][0]}x{c[0][1]}x{c[0][2]}_n{c[4]}_nc{c[5]}")
def test_symmetric_apply_matches_full_oracle(case, variant):
    dims, bc, omega, h, n, n_c = case
    nx, ny, nz = dims
    rng = np.random.default_rng(23)
    psi = rng.standard_normal((n, nz, ny, nx))
    occ = np.linspace(2.0, 1e-6, n)                      # distinct occupations: a swapped occ_j/occ_k would show
    o = orc.make_plan(nx, ny, nz, h, bc, 12, omega)
    vx_o, e_o, ex_o = orc.exx_apply(o, psi, occ, psi, occ)
    plan = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=64, device=0)
    plan.set_variant(variant)
    d_psi, d_occ = torch.from_numpy(psi).cuda(), torch.from_numpy(occ).cuda()
    tma0 = plan.tma_launch_count
    vx, e_k, ex = plan.apply_symmetric(d_psi, d_occ, n_c=n_c)
    torch.cuda.synchronize()
    two_sided = variant == exx.VARIANT_FUSED_DMMA and min(dims) >= 34
    assert plan.last_solve_count == _expected_solves(n, n_c, _nk_min(*dims) if two_sided else 1)
    if two_sided:       # six TMA-staged launches per batch (no streaming accumulate kernel) + zero fills and the energy
        assert plan.tma_launch_count - tma0 == plan.last_launch_count - 4 and (plan.last_launch_count - 4) % 6 == 0
    assert n * (n + 1) // 2 <= plan.last_solve_count < n * n or n == 1
    assert _rel(vx.cpu().numpy(), vx_o) < TOL
    assert np.abs(e_k.cpu().numpy() - e_o).max() < TOL * np.abs(e_o).max()
    assert abs(ex.item() - ex_o) < TOL * abs(ex_o)
    # and against the library's own full apply
    vx_f, _, ex_f = plan.apply(d_psi, d_occ, d_psi, d_occ, n_c=n_c)
    torch.cuda.synchronize()
    assert plan.last_solve_count == n * n
    assert _rel(vx.cpu().numpy(), vx_f.cpu().numpy()) < 1e-12
    if two_sided:
        # with both sides of the accumulate fused into the x-backward pass every vx_m receives its terms in
        # ascending partner order (target side j <= m first, orbital side k > m after), each term formed by the same
        # instructions from the same phi bits as in the full apply: the two results are bitwise equal
        assert torch.equal(vx, vx_f), f"max abs diff {float((vx - vx_f).abs().max()):.3e}"
        assert ex.item() == ex_f.item()
    plan.close()


# The unfused route of the pair-symmetric apply on grids where the two-sided fused accumulate COULD run: the streaming
# k_accumulate (sym) + k_accumulate_transposed pair behind mode products that still run in symmetric mode order for y and z.
# It is taken when fusion bit 1 is off (mask 13) and when a buffer is not 16-byte aligned (TMA cannot address it).  Either
# way exx_apply_symmetric shapes its blocks with nk_min = 1, so nk >= 2 only where the whole block is one j-chunk.
@pytest.mark.parametrize("how", ["fusion13", "psi_offset_8_bytes"])
@pytest.mark.parametrize("case", [((40, 36, 34), (0, 0, 1), 0.106, 0.3, 21, 16), ((36, 40, 44), (1, 0, 0), 0.0, 0.3, 11, 5)],
                         ids=lambda c: f"{c[0][0]}x{c[0][1]}x{c[0][2]}_n{c[4]}_nc{c[5]}")
def test_symmetric_apply_unfused_route_on_symmetric_capable_grids(case, how):
    dims, bc, omega, h, n, n_c = case
    nx, ny, nz = dims
    rng = np.random.default_rng(29)
    psi = rng.standard_normal((n, nz, ny, nx))
    occ = np.linspace(2.0, 1e-6, n)
    o = orc.make_plan(nx, ny, nz, h, bc, 12, omega)
    vx_o, e_o, ex_o = orc.exx_apply(o, psi, occ, psi, occ)
    plan = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=64, device=0)
    d_occ = torch.from_numpy(occ).cuda()
    if how == "fusion13":
        plan.set_fusion(13)
        d_psi = torch.from_numpy(psi).cuda()
    else:
        flat = torch.empty(psi.size + 1, dtype=torch.float64, device="cuda")
        d_psi = flat[1:].view(n, nz, ny, nx)
        d_psi.copy_(torch.from_numpy(psi))
        assert d_psi.data_ptr() % 16 == 8
    vx, e_k, ex = plan.apply_symmetric(d_psi, d_occ, n_c=n_c)
    torch.cuda.synchronize()
    assert plan.last_solve_count == _expected_solves(n, n_c, 1)      # nk_min = 1: the two-sided pass was not chosen
    assert _rel(vx.cpu().numpy(), vx_o) < TOL
    assert np.abs(e_k.cpu().numpy() - e_o).max() < TOL * np.abs(e_o).max()
    assert abs(ex.item() - ex_o) < TOL * abs(ex_o)
    plan.close()


def test_symmetric_on_config2_full_size():
    w = wl.WORKLOADS[2]
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    o = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    vx_o, e_o, ex_o = orc.exx_apply(o, psi.numpy(), occ.numpy(), psi.numpy(), occ.numpy())
    plan = exx.Plan.for_workload(w, device=0)
    vx, e_k, ex = plan.apply_symmetric(psi.cuda(), occ.cuda(), n_c=128)
    torch.cuda.synchronize()
    assert plan.last_solve_count == _expected_solves(w.n_orb, 128, _nk_min(w.nx, w.ny, w.nz)) < 0.6 * w.n_orb ** 2
    assert _rel(vx.cpu().numpy(), vx_o) < TOL
    assert abs(ex.item() - ex_o) < TOL * abs(ex_o)
    plan.close()


def test_symmetric_empty_and_errors():
    plan = exx.Plan(8, 8, 8, 0.5, (0, 0, 0), 12, 0.106, max_batch=4, device=0)
    z = torch.zeros((0, 8, 8, 8), dtype=torch.float64, device="cuda")
    vx, e_k, ex = plan.apply_symmetric(z, torch.zeros(0, dtype=torch.float64, device="cuda"))
    torch.cuda.synchronize()
    assert vx.shape[0] == 0 and ex.item() == 0.0 and plan.last_solve_count == 0
    x = torch.zeros((2, 8, 8, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(exx.ExxError) as ei:
        plan.apply_symmetric(x, torch.ones(2, dtype=torch.float64, device="cuda"), vx=x)
    assert ei.value.status == 6
    plan.close()
