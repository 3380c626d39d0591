"""C-ABI host-side checks (CPU only): the library loads, exports every symbol include/exx.h declares,
validates arguments, and its own planner (FD matrices + Jacobi + multiplier table, no code shared with
the oracle) agrees with the oracle's numpy/LAPACK planner.  No compute call is made."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import __graft_entry__ as ge
from oracle import exx_oracle as orc
from paper_2501_16572_b200 import exx

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    ge.build()
    return exx.load_library()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "exx.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    names = set(re.findall(r"\b(exx_[a-z_]+)\s*\(", header))
    assert {"exx_plan_create", "exx_plan_destroy", "exx_apply", "exx_poisson_solve", "exx_apply_host",
            "exx_plan_workspace_bytes", "exx_status_string"} <= names
    for n in names:
        assert hasattr(lib, n), n
    assert b"sm_100a" in lib.exx_version()


def test_argument_validation_without_gpu(lib):
    h = C.c_void_p()
    bc = (C.c_int * 3)(0, 0, 0)
    bad = [
        dict(nx=0), dict(h=0.0), dict(h=-1.0), dict(order=3), dict(order=0), dict(max_batch=0),
    ]
    for kw in bad:
        a = dict(nx=8, ny=8, nz=8, h=0.5, order=12, omega=0.0, max_batch=4)
        a.update(kw)
        st = lib.exx_plan_create(C.byref(h), a["nx"], a["ny"], a["nz"], a["h"], bc, a["order"], a["omega"],
                                 a["max_batch"], -1)
        assert st == 1, kw
        assert not h.value
    bc_bad = (C.c_int * 3)(0, 2, 0)
    assert lib.exx_plan_create(C.byref(h), 8, 8, 8, 0.5, bc_bad, 12, 0.0, 4, -1) == 1
    assert lib.exx_plan_create(None, 8, 8, 8, 0.5, bc, 12, 0.0, 4, -1) == 1
    for s in range(7):
        assert lib.exx_status_string(s).startswith(b"EXX_")


def test_host_only_plan_refuses_compute_loudly(lib):
    p = exx.Plan(8, 6, 5, 0.5, (0, 0, 1), 12, 0.106, max_batch=4, device=-1)
    assert p.workspace_bytes(4) == 2 * 8 * 240 * 4
    assert p.workspace_bytes(5) == 0          # > max_batch
    assert p.workspace_bytes(0) == 2 * 8 * 240 * 4  # default clamps to max_batch
    dummy = C.c_void_p(1 << 20)
    st = lib.exx_poisson_solve(p._h, dummy, dummy, 1, 1, dummy, 1 << 30, None)
    assert st == 3 and b"EXX_ERR_CUDA" in lib.exx_status_string(st)   # no CPU fallback
    st = lib.exx_apply(p._h, dummy, dummy, 1, dummy, None, 1, C.c_void_p(1 << 28), None, None, 1, C.c_void_p(1 << 29),
                       1 << 20, None)
    assert st == 3
    with pytest.raises(exx.ExxError):
        p.set_variant(7)
    p.close()


def test_energy_static_validates_before_touching_a_device(lib):
    """exx_energy_static (the entry point for callers that cannot allocate device memory): argument errors and the
    fixed capacity of its in-library scratch array are reported before any CUDA call, so they can be checked without a
    GPU; with valid arguments and no device the call fails loudly (there is no CPU fallback)."""
    d = C.c_void_p(1 << 20)
    f = lib.exx_energy_static
    assert f(d, d, d, exx.ENERGY_STATIC_MAX_TGT + 1, 10, 1.0, d, d, None) == 7           # EXX_ERR_LIMIT
    assert b"EXX_ERR_LIMIT" in lib.exx_status_string(7) and b"4096" in lib.exx_status_string(7)
    assert f(d, d, d, -1, 10, 1.0, d, d, None) == 1                                       # n_tgt < 0
    assert f(d, d, d, 2, 0, 1.0, d, d, None) == 1                                         # n_points < 1
    assert f(d, d, d, 2, 10, 0.0, d, d, None) == 1                                        # dv <= 0
    assert f(None, d, d, 2, 10, 1.0, d, d, None) == 1                                     # missing input
    assert f(d, d, None, 2, 10, 1.0, d, d, None) == 1                                     # E_x without occupations
    assert f(d, d, d, 2, 10, 1.0, None, None, None) == 0                                  # nothing asked for: a no-op
    import torch
    if not torch.cuda.is_available():
        st = f(d, d, d, 2, 10, 1.0, d, d, None)
        assert st == 3 and b"EXX_ERR_CUDA" in lib.exx_status_string(st)


@pytest.mark.parametrize("dims,bc,omega,h", [((16, 16, 16), (0, 0, 0), 0.0, 0.5), ((12, 10, 30), (0, 0, 1), 0.106, 0.25),
                                             ((48, 48, 48), (0, 0, 0), 0.106, 0.25), ((7, 9, 5), (1, 0, 1), 0.106, 0.3),
                                             ((120, 60, 1), (1, 0, 0), 0.106, 0.2)])
def test_library_planner_agrees_with_oracle_planner(lib, dims, bc, omega, h):
    nx, ny, nz = dims
    p = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=4, device=-1)
    o = orc.make_plan(nx, ny, nz, h, bc, 12, omega)
    scale = abs(orc.fd_weights(12, h)[0])
    for ax, n in enumerate(dims):
        lam, V = p.get_axis(ax)
        assert np.allclose(lam, o.lam[ax], rtol=0, atol=2e-13 * scale)
        assert np.allclose(V.T @ V, np.eye(n), atol=1e-13)
        K = orc.second_derivative_matrix(n, h, bc[ax], 12)
        assert np.allclose(K @ V, V * lam[None, :], rtol=0, atol=5e-13 * scale)
    # eigenvalue sums are basis independent => tables must agree entry by entry (incl. the zero-mode rule)
    m = p.get_multiplier()
    assert m.shape == o.mult.shape
    assert np.allclose(m, o.mult, rtol=1e-10, atol=0)
    if all(b == 0 for b in bc):
        assert m[-1, -1, -1] == (0.0 if omega <= 0 else pytest.approx(np.pi / omega ** 2, rel=1e-14))
    p.close()


@pytest.mark.parametrize("dims,bc,h", [((16, 12, 9), (0, 0, 1), 0.3), ((48, 60, 120), (0, 0, 1), 0.25), ((120, 96, 7), (0, 0, 0), 0.2),
                                       ((5, 13, 126), (1, 1, 0), 0.4), ((1, 2, 3), (0, 0, 0), 0.5), ((2, 4, 128), (1, 1, 1), 0.5)])
def test_reflection_adapted_eigenbasis(lib, dims, bc, h):
    """exx_plan_get_axis_symmetric (the basis the fused z pass contracts with): the same eigenpairs as the
    oracle's matrix, every vector EXACTLY even or odd under z -> mir(z), even block first with one vector per z <= mir(z),
    and the spectral projector of every eigenvalue cluster equal to the one of the plain basis (so f(L) is unchanged)."""
    nx, ny, nz = dims
    p = exx.Plan(nx, ny, nz, h, bc, 12, 0.106, max_batch=4, device=-1)
    scale = abs(orc.fd_weights(12, h)[0])
    for ax, n in enumerate(dims):
        lam0, V0 = p.get_axis(ax)
        lam, V, ne = p.get_axis_symmetric(ax)
        mir = n - 1 - np.arange(n)
        assert ne == int(np.sum(np.arange(n) <= mir))
        assert np.all(V[mir, :ne] == V[:, :ne]) and np.all(V[mir, ne:] == -V[:, ne:])      # exact parity
        assert np.all(np.diff(lam[:ne]) >= -1e-12 * scale) and np.all(np.diff(lam[ne:]) >= -1e-12 * scale)
        assert np.allclose(np.sort(lam), lam0, rtol=0, atol=1e-12 * scale)
        assert np.allclose(V.T @ V, np.eye(n), atol=1e-12)      # parity parts are renormalised: a decade above Jacobi's own
        K = orc.second_derivative_matrix(n, h, bc[ax], 12)
        assert np.allclose(K @ V, V * lam[None, :], rtol=0, atol=1e-12 * scale)
        # any function of K is the same in both bases
        f = lambda l: np.exp(l / scale)
        assert np.allclose((V * f(lam)[None, :]) @ V.T, (V0 * f(lam0)[None, :]) @ V0.T, rtol=0, atol=1e-12)
    p.close()


@pytest.mark.parametrize("dims,bc,theta", [((16, 12, 9), (0, 0, 1), (0.7, -2.1, 0.5)), ((48, 48, 48), (0, 0, 0), (np.pi, 0.0, 1.0)),
                                           ((7, 60, 5), (1, 0, 0), (0.3, np.pi / 2, -np.pi))])
@pytest.mark.parametrize("form", [0, 1], ids=["real_form", "embedded"])
def test_bloch_planner_agrees_with_bloch_oracle(lib, dims, bc, theta, form):
    """exx_plan_create_bloch (form 0: the real form K' = U^H K U = W Lambda W^T through the reflection butterfly U, Jacobi,
    V = U W) and exx_plan_create_bloch_form(EMBEDDED) (real-symmetric embedding + Jacobi + complex Gram-Schmidt) against
    numpy's Hermitian eigh on the oracle's matrix: eigenvalues, unitarity, K V = V Lambda, and the multiplier table."""
    from oracle import bloch_oracle as blo
    nx, ny, nz = dims
    h, omega = 0.3, 0.106
    p = exx.Plan(nx, ny, nz, h, bc, 12, omega, max_batch=4, device=-1, theta=theta, bloch_form=form)
    o = blo.make_plan(nx, ny, nz, h, bc, 12, omega, theta)
    scale = abs(blo.fd_weights(12, h)[0])
    for ax, n in enumerate(dims):
        lam, V = p.get_axis_bloch(ax)
        assert np.allclose(lam, o.lam[ax], rtol=0, atol=5e-13 * scale)
        assert np.allclose(V.conj().T @ V, np.eye(n), atol=1e-12)
        K = blo.bloch_second_derivative_matrix(n, h, bc[ax], 12, theta[ax])
        assert np.allclose(K @ V, V * lam[None, :], rtol=0, atol=2e-12 * scale)
        if bc[ax] == 1 or theta[ax] == 0.0:
            assert np.all(V.imag == 0.0)           # real axis: the real planner was used
            p.get_axis_symmetric(ax)               # ... and it still has its reflection-adapted basis
        else:
            # an axis with a phase has no reflection-adapted real basis, in either form (in the real form h_V holds W of
            # K' = U^H K U, not eigenvectors of K): exx_plan_get_axis_symmetric says INVALID_ARG, as exx.h documents
            with pytest.raises(exx.ExxError) as err:
                p.get_axis_symmetric(ax)
            assert err.value.status == 1
    assert np.allclose(p.get_multiplier(), o.mult, rtol=1e-10, atol=0)
    # the real entry points refuse a complex plan
    dummy = C.c_void_p(1 << 20)
    assert lib.exx_poisson_solve(p._h, dummy, dummy, 1, 1, dummy, 1 << 30, None) == 1
    assert p._lib.exx_plan_workspace_bytes_bloch(p._h, 4) == 6 * 8 * nx * ny * nz * 4
    p.close()
