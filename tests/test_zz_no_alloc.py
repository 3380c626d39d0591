"""exx_energy_static, the one entry point of libexx.so that allocates nothing, against the energy outputs of exx_apply.

Why the entry point exists: some users of the library cannot call cudaMalloc when they need the exchange energy.  A
host code that gave the whole card to its own memory arena at start-up gets an out-of-memory error from any later
allocation, and a caller that keeps several streams busy cannot afford the device-wide stall that comes with
cudaMalloc / cudaFree.  For them the energy step (e_k = h^3 <tgt_k, vx_k>, E_x = 1/2 sum_k occ_k e_k) is offered with
its scratch -- 64 block sums per target -- in a fixed 2 MiB array inside the library, shared by every call on a device.

What is checked, on two calls in a row so that whatever the first call leaves in the shared array is there when the
second one runs: each call's e_k and E_x equal those exx_apply computed for the same vx (existing path: plan-owned
scratch from cudaMalloc), within the 1e-10 relative tolerance of the parity tests; the second call has fewer targets
and different data than the first.  The size limit answers with EXX_ERR_LIMIT before anything is enqueued.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here hides no other test) and does
not depend on what ran before it: the first call in a process performs the entry point's per-device set-up."""
import numpy as np
import pytest
import torch

from paper_2501_16572_b200 import exx, workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as ge
    ge.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"


def _existing_path(plan, psi, occ, tgt, occ_t):
    """exx_apply with its own energy outputs: (vx, e_k, E_x) on the device."""
    vx, e_k, ex = plan.apply(psi, occ, tgt, occ_t)
    torch.cuda.synchronize()
    return vx, e_k, ex


def _static_path(tgt, vx, occ_t, dv):
    """The no-allocation entry point; the outputs are the caller's, poisoned so that a skipped write shows."""
    e_k = torch.full((tgt.shape[0],), float("nan"), dtype=torch.float64, device=tgt.device)
    ex = torch.full((), float("nan"), dtype=torch.float64, device=tgt.device)
    exx.energy_static(tgt, vx, occ_t, dv, e_k, ex)
    torch.cuda.synchronize()
    return e_k, ex


def _close(a, b):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    return float(np.abs(a - b).max()) <= TOL * float(np.abs(b).max())


def test_energy_static_matches_exx_apply_on_two_calls_in_a_row():
    dev = torch.device("cuda", 0)
    w = wl.WORKLOADS[1]                                   # 16^3, 8 orbitals, all of them targets
    psi, occ, tgt, occ_t = (t.to(dev) for t in wl.make_inputs(w, "cpu"))
    plan = exx.Plan.for_workload(w, device=0)
    dv = w.h * w.h * w.h

    # first call: all 8 targets
    vx1, e1, ex1 = _existing_path(plan, psi, occ, tgt, occ_t)
    s_e1, s_ex1 = _static_path(tgt, vx1, occ_t, dv)
    assert _close(s_e1, e1) and _close(s_ex1, ex1)

    # second call, straight after: 3 other targets (random, not orbitals), fractional weights; the array still holds
    # the first call's 8 x 64 block sums
    g = torch.Generator().manual_seed(7)
    tgt2 = torch.randn((3, w.nz, w.ny, w.nx), dtype=torch.float64, generator=g).to(dev)
    occ2 = torch.tensor([0.25, 1.5, 2.0], dtype=torch.float64, device=dev)
    vx2, e2, ex2 = _existing_path(plan, psi, occ, tgt2, occ2)
    s_e2, s_ex2 = _static_path(tgt2, vx2, occ2, dv)
    assert _close(s_e2, e2) and _close(s_ex2, ex2)
    assert not _close(s_ex2, ex1)                          # the two calls really had different answers

    # and the first inputs once more give the first answer again
    s_e3, s_ex3 = _static_path(tgt, vx1, occ_t, dv)
    assert torch.equal(s_e3, s_e1) and torch.equal(s_ex3, s_ex1)
    plan.close()


def test_energy_static_rejects_more_targets_than_its_array_holds():
    dev = torch.device("cuda", 0)
    n = exx.ENERGY_STATIC_MAX_TGT + 1
    tgt = torch.ones((n, 4), dtype=torch.float64, device=dev)
    occ = torch.ones(n, dtype=torch.float64, device=dev)
    e_k = torch.full((n,), -7.0, dtype=torch.float64, device=dev)
    ex = torch.full((), -7.0, dtype=torch.float64, device=dev)
    with pytest.raises(exx.ExxError) as err:
        exx.energy_static(tgt, tgt, occ, 1.0, e_k, ex)
    assert err.value.status == 7 and "EXX_ERR_LIMIT" in str(err.value) and "4096" in str(err.value)
    torch.cuda.synchronize()
    assert float(ex) == -7.0 and bool((e_k == -7.0).all())  # nothing was enqueued
    # exactly at the limit it runs: <1, 1> over 4 points, dv = 1
    exx.energy_static(tgt[:n - 1], tgt[:n - 1], occ[:n - 1], 1.0, e_k[:n - 1], ex)
    torch.cuda.synchronize()
    assert bool((e_k[:n - 1] == 4.0).all()) and float(ex) == 0.5 * 4.0 * (n - 1)


def test_energy_static_on_the_two_plane_complex_sets_of_the_bloch_variant():
    """n_points = 2 N: a complex function is a real plane followed by an imaginary plane, and the plain dot product over
    both planes is Re <tgt, vx> -- the e_k exx_apply_bloch returns (its existing path, same tolerance)."""
    dev = torch.device("cuda", 0)
    nx, ny, nz, h = 16, 12, 10, 0.35
    plan = exx.Plan(nx, ny, nz, h, (0, 0, 1), 12, 0.106, max_batch=8, device=0, theta=(0.6, -1.0, 0.0))
    g = torch.Generator().manual_seed(11)
    psi = torch.randn((5, 2, nz, ny, nx), dtype=torch.float64, generator=g).to(dev)
    tgt = torch.randn((3, 2, nz, ny, nx), dtype=torch.float64, generator=g).to(dev)
    occ = torch.linspace(2.0, 0.1, 5, dtype=torch.float64).to(dev)
    vx, e_k = plan.apply_bloch(psi, occ, tgt, n_c=4)
    torch.cuda.synchronize()
    s_e = torch.full((3,), float("nan"), dtype=torch.float64, device=dev)
    exx.energy_static(tgt, vx, None, h * h * h, s_e, None)      # no occupations: e_k only
    torch.cuda.synchronize()
    assert _close(s_e, e_k)
    plan.close()
