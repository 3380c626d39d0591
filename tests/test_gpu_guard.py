"""Out-of-bounds guard (compute-sanitizer is not available on the GPU pool): every output buffer and the workspace are
carved out of a larger canary-filled allocation; after each call the canaries on both sides must be intact.  Ragged
sizes (not multiples of the 8/16/32/64 tile edges), all entry points."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2501_16572_b200 import exx

pytestmark = pytest.mark.gpu
CANARY = -7.25e300
PAD = 4096  # doubles on each side


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as ge
    ge.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"


class Guarded:
    def __init__(self, shape):
        n = int(np.prod(shape))
        self.raw = torch.full((n + 2 * PAD,), CANARY, dtype=torch.float64, device="cuda")
        self.t = self.raw[PAD:PAD + n].view(*shape)

    def intact(self):
        return bool((self.raw[:PAD] == CANARY).all() and (self.raw[-PAD:] == CANARY).all())


def _guarded_workspace(plan, nbytes):
    g = Guarded((nbytes // 8 + 2,))
    plan._ws = g.t.view(torch.uint8)[:nbytes]        # the binding hands this tensor to the library as the workspace
    return g


GRIDS = [((20, 12, 9), (0, 1, 0)), ((13, 17, 11), (1, 1, 1)), ((34, 10, 70), (0, 0, 1)), ((16, 16, 16), (0, 0, 0))]


@pytest.mark.parametrize("dims,bc", GRIDS)
def test_real_entry_points_stay_inside_their_buffers(dims, bc):
    nx, ny, nz = dims
    rng = np.random.default_rng(3)
    plan = exx.Plan(nx, ny, nz, 0.3, bc, 12, 0.106, max_batch=16, device=0)
    n = 7
    psi = torch.from_numpy(rng.standard_normal((n, nz, ny, nx))).cuda()
    occ = torch.linspace(2.0, 0.1, n, dtype=torch.float64).cuda()
    ws = _guarded_workspace(plan, plan.workspace_bytes(5))
    vx = Guarded((n, nz, ny, nx))
    plan.apply(psi, occ, psi, occ, vx=vx.t, n_c=5)
    torch.cuda.synchronize()
    assert vx.intact() and ws.intact() and torch.isfinite(vx.t).all()
    vs = Guarded((n, nz, ny, nx))
    plan.apply_symmetric(psi, occ, vx=vs.t, n_c=5)
    torch.cuda.synchronize()
    assert vs.intact() and ws.intact()
    assert float((vs.t - vx.t).abs().max()) < 1e-12 * float(vx.t.abs().max())
    out = Guarded((3, nz, ny, nx))
    plan.poisson_solve(psi[:3].contiguous(), out=out.t, n_c=2)
    torch.cuda.synchronize()
    assert out.intact() and ws.intact()
    # ACE: xi, M and the trial output
    aws = Guarded((plan.ace_workspace_bytes(n, 3) // 8 + 2,))
    plan._aws = aws.t.view(torch.uint8)[:plan.ace_workspace_bytes(n, 3)]
    xi = Guarded((n, nz, ny, nx))
    plan.ace_build(psi, vx.t, xi=xi.t)
    o2 = Guarded((3, nz, ny, nx))
    plan.ace_apply(xi.t, psi[:3].contiguous(), out=o2.t)
    torch.cuda.synchronize()
    assert xi.intact() and o2.intact() and aws.intact() and torch.isfinite(o2.t).all()
    plan.close()


@pytest.mark.parametrize("dims,bc,theta", [((20, 12, 10), (0, 0, 1), (0.5, 0.3, 0.0)), ((16, 16, 16), (0, 0, 0), (0.9, -0.4, 2.0)),
                                           ((13, 8, 10), (0, 0, 0), (1.0, 0.0, 0.7))])
def test_bloch_entry_points_stay_inside_their_buffers(dims, bc, theta):
    nx, ny, nz = dims
    rng = np.random.default_rng(5)
    plan = exx.Plan(nx, ny, nz, 0.3, bc, 12, 0.106, max_batch=8, device=0, theta=theta)
    psi = torch.from_numpy(rng.standard_normal((5, 2, nz, ny, nx))).cuda()
    occ = torch.ones(5, dtype=torch.float64).cuda()
    nbytes = int(plan._lib.exx_plan_workspace_bytes_bloch(plan._h, 4))
    ws = _guarded_workspace(plan, nbytes)
    vx = Guarded((2, 2, nz, ny, nx))
    plan.apply_bloch(psi, occ, psi[:2].contiguous(), vx=vx.t, n_c=4)
    out = Guarded((3, 2, nz, ny, nx))
    plan.poisson_solve_bloch(psi[:3].contiguous(), out=out.t, n_c=4)
    torch.cuda.synchronize()
    assert vx.intact() and out.intact() and ws.intact() and torch.isfinite(vx.t).all() and torch.isfinite(out.t).all()
    plan.close()
