"""Thin ctypes binding over libexx.so (include/exx.h).  Argument marshalling only: every step of
the hot path runs in the library's CUDA kernels.  torch is used for device memory and streams.

There is no CPU fallback: if libexx.so is missing or a call fails, an :class:`ExxError` is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))

EXX_OK = 0
BC_PERIODIC, BC_DIRICHLET = 0, 1
VARIANT_FUSED_DMMA, VARIANT_REFERENCE, VARIANT_CPASYNC = 0, 1, 2

_lib = None


class ExxError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = load_library().exx_status_string(status).decode()
        super().__init__(f"{where}: {msg}")


def lib_path() -> str:
    return os.path.join(HERE, "libexx.so")


def load_library():
    """dlopen libexx.so (built in-tree by ``paper_2501_16572_b200.build``); fail loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise RuntimeError(
            f"{path} not found: build it with `python -m paper_2501_16572_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.c_void_p, C.POINTER(C.c_int)
    lib.exx_plan_create.restype = C.c_int
    lib.exx_plan_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_double, ip, C.c_int,
                                    C.c_double, C.c_int, C.c_int]
    lib.exx_plan_destroy.restype = C.c_int
    lib.exx_plan_destroy.argtypes = [vp]
    lib.exx_plan_set_variant.restype = C.c_int
    lib.exx_plan_set_variant.argtypes = [vp, C.c_int]
    lib.exx_plan_workspace_bytes.restype = C.c_size_t
    lib.exx_plan_workspace_bytes.argtypes = [vp, C.c_int]
    lib.exx_plan_get_axis.restype = C.c_int
    lib.exx_plan_get_axis.argtypes = [vp, C.c_int, dp, dp]
    lib.exx_plan_get_multiplier.restype = C.c_int
    lib.exx_plan_get_multiplier.argtypes = [vp, dp]
    lib.exx_plan_get_axis_symmetric.restype = C.c_int
    lib.exx_plan_get_axis_symmetric.argtypes = [vp, C.c_int, dp, dp, C.POINTER(C.c_int)]
    lib.exx_plan_executed_flops_per_solve.restype = C.c_double
    lib.exx_plan_executed_flops_per_solve.argtypes = [vp]
    lib.exx_plan_executed_flops_per_symmetric_solve.restype = C.c_double
    lib.exx_plan_executed_flops_per_symmetric_solve.argtypes = [vp]
    lib.exx_poisson_solve.restype = C.c_int
    lib.exx_poisson_solve.argtypes = [vp, dp, dp, C.c_int, C.c_int, vp, C.c_size_t, vp]
    lib.exx_poisson_solve_nonbatch.restype = C.c_int
    lib.exx_poisson_solve_nonbatch.argtypes = [vp, dp, dp, C.c_int, vp, C.c_size_t, vp]
    lib.exx_apply.restype = C.c_int
    lib.exx_apply.argtypes = [vp, dp, dp, C.c_int, dp, dp, C.c_int, dp, dp, dp, C.c_int, vp, C.c_size_t, vp]
    lib.exx_apply_symmetric.restype = C.c_int
    lib.exx_apply_symmetric.argtypes = [vp, dp, dp, C.c_int, dp, dp, dp, C.c_int, vp, C.c_size_t, vp]
    lib.exx_plan_last_solve_count.restype = C.c_longlong
    lib.exx_plan_last_solve_count.argtypes = [vp]
    lib.exx_apply_host.restype = C.c_int
    lib.exx_apply_host.argtypes = [vp, dp, dp, C.c_int, dp, C.c_int, dp, C.c_int, dp, dp, dp, C.c_int]
    lib.exx_plan_last_launch_count.restype = C.c_longlong
    lib.exx_plan_last_launch_count.argtypes = [vp]
    lib.exx_plan_tma_launch_count.restype = C.c_longlong
    lib.exx_plan_tma_launch_count.argtypes = [vp]
    lib.exx_plan_set_lanes.restype = C.c_int
    lib.exx_plan_set_lanes.argtypes = [vp, C.c_int]
    lib.exx_plan_set_accumulate.restype = C.c_int
    lib.exx_plan_set_accumulate.argtypes = [vp, C.c_int]
    lib.exx_plan_get_lanes.restype = C.c_int
    lib.exx_plan_get_lanes.argtypes = [vp]
    lib.exx_plan_set_fusion.restype = C.c_int
    lib.exx_plan_set_fusion.argtypes = [vp, C.c_int]
    lib.exx_plan_get_fusion.restype = C.c_int
    lib.exx_plan_get_fusion.argtypes = [vp]
    lib.exx_ace_workspace_bytes.restype = C.c_size_t
    lib.exx_ace_workspace_bytes.argtypes = [vp, C.c_int, C.c_int]
    lib.exx_ace_build.restype = C.c_int
    lib.exx_ace_build.argtypes = [vp, dp, dp, C.c_int, dp, dp, vp, vp, C.c_size_t, vp]
    lib.exx_ace_apply.restype = C.c_int
    lib.exx_ace_apply.argtypes = [vp, dp, C.c_int, dp, C.c_int, dp, vp, C.c_size_t, vp]
    lib.exx_ace_workspace_bytes_bloch.restype = C.c_size_t
    lib.exx_ace_workspace_bytes_bloch.argtypes = [vp, C.c_int, C.c_int]
    lib.exx_ace_build_bloch.restype = C.c_int
    lib.exx_ace_build_bloch.argtypes = [vp, dp, dp, C.c_int, dp, dp, vp, vp, C.c_size_t, vp]
    lib.exx_ace_apply_bloch.restype = C.c_int
    lib.exx_ace_apply_bloch.argtypes = [vp, dp, C.c_int, dp, C.c_int, dp, vp, C.c_size_t, vp]
    lib.exx_plan_create_bloch.restype = C.c_int
    lib.exx_plan_create_bloch.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_double, ip, C.c_int,
                                          C.c_double, C.POINTER(C.c_double), C.c_int, C.c_int]
    lib.exx_plan_create_bloch_form.restype = C.c_int
    lib.exx_plan_create_bloch_form.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_double, ip, C.c_int,
                                               C.c_double, C.POINTER(C.c_double), C.c_int, C.c_int, C.c_int]
    lib.exx_plan_workspace_bytes_bloch.restype = C.c_size_t
    lib.exx_plan_workspace_bytes_bloch.argtypes = [vp, C.c_int]
    lib.exx_poisson_solve_bloch.restype = C.c_int
    lib.exx_poisson_solve_bloch.argtypes = [vp, dp, dp, C.c_int, C.c_int, vp, C.c_size_t, vp]
    lib.exx_apply_bloch.restype = C.c_int
    lib.exx_apply_bloch.argtypes = [vp, dp, dp, C.c_int, dp, C.c_int, dp, C.c_int, dp, C.c_int, vp, C.c_size_t, vp]
    lib.exx_plan_get_axis_bloch.restype = C.c_int
    lib.exx_plan_get_axis_bloch.argtypes = [vp, C.c_int, dp, dp, dp]
    lib.exx_status_string.restype = C.c_char_p
    lib.exx_status_string.argtypes = [C.c_int]
    lib.exx_plan_set_profiling.restype = C.c_int
    lib.exx_plan_set_profiling.argtypes = [vp, C.c_int]
    lib.exx_plan_get_profile.restype = C.c_int
    lib.exx_plan_get_profile.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    lib.exx_plan_get_profile_passes.restype = C.c_int
    lib.exx_plan_get_profile_passes.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong), C.POINTER(C.c_double)]
    lib.exx_probe_fp64_peak.restype = C.c_int
    lib.exx_probe_fp64_peak.argtypes = [C.c_int, C.c_int, C.c_double, C.POINTER(C.c_double)]
    lib.exx_energy_static.restype = C.c_int
    lib.exx_energy_static.argtypes = [dp, dp, dp, C.c_int, C.c_longlong, C.c_double, dp, dp, vp]
    lib.exx_version.restype = C.c_char_p
    lib.exx_version.argtypes = []
    _lib = lib
    return lib


def _check(status: int, where: str):
    if status != EXX_OK:
        raise ExxError(status, where)


def _dev_ptr(t: torch.Tensor | None, device: torch.device, what: str):
    if t is None:
        return None
    if t.dtype != torch.float64 or not t.is_contiguous():
        raise ValueError(f"{what}: need a contiguous float64 tensor")
    if t.device != device:
        raise ValueError(f"{what}: tensor is on {t.device}, plan is on {device}")
    return C.c_void_p(t.data_ptr())


def _host_ptr(t, what: str):
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        if t.dtype != np.float64 or not t.flags.c_contiguous:
            raise ValueError(f"{what}: need a C-contiguous float64 array")
        return C.c_void_p(t.ctypes.data)
    if t.dtype != torch.float64 or not t.is_contiguous() or t.device.type != "cpu":
        raise ValueError(f"{what}: need a contiguous float64 host tensor")
    return C.c_void_p(t.data_ptr())


def probe_fp64_peak(kind: int, device: int = 0, seconds: float = 1.0) -> float:
    """exx_probe_fp64_peak: sustained TFLOP/s of a DFMA (kind 0) or DMMA (kind 1) issue loop."""
    out = C.c_double(0.0)
    _check(load_library().exx_probe_fp64_peak(kind, device, seconds, C.byref(out)), "exx_probe_fp64_peak")
    return out.value


ENERGY_STATIC_MAX_TGT = 4096     # EXX_ENERGY_STATIC_MAX_TGT (include/exx.h)


def energy_static(tgt: torch.Tensor, vx: torch.Tensor, occ_tgt: torch.Tensor | None, dv: float,
                  ex_k: torch.Tensor | None, ex: torch.Tensor | None, stream: torch.cuda.Stream | None = None) -> None:
    """exx_energy_static: ex_k[k] = dv <tgt[k], vx[k]>, ex = 1/2 sum_k occ_tgt[k] ex_k[k], written into the tensors the
    caller passes (either may be None).  Meant for callers that cannot allocate on the GPU -- all device memory already
    given to their own arena, or a multi-stream loop that a cudaMalloc would stall: the library call needs no plan and
    no workspace and allocates nothing (its block sums go to a fixed 2 MiB array inside libexx.so), which is why this
    wrapper takes the outputs instead of creating them.  At most ENERGY_STATIC_MAX_TGT targets per call (ExxError with
    EXX_ERR_LIMIT beyond).  Runs on the tensors' device, which is made current for the call; calls that overlap on that
    GPU race on the shared array, so keep them on one stream."""
    n_tgt = tgt.shape[0]
    dev = tgt.device
    n_points = tgt.numel() // n_tgt if n_tgt else max(1, vx.numel())
    if vx.numel() != tgt.numel():
        raise ValueError("tgt and vx must hold the same number of elements")
    for t, n, what in ((occ_tgt, n_tgt, "occ_tgt"), (ex_k, n_tgt, "ex_k"), (ex, 1, "ex")):
        if t is not None and t.numel() != n:
            raise ValueError(f"{what}: expected {n} elements, got {t.numel()}")
    with torch.cuda.device(dev):
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        st = load_library().exx_energy_static(_dev_ptr(tgt, dev, "tgt"), _dev_ptr(vx, dev, "vx"),
                                              _dev_ptr(occ_tgt, dev, "occ_tgt"), n_tgt, n_points, float(dv),
                                              _dev_ptr(ex_k, dev, "ex_k"), _dev_ptr(ex, dev, "ex"),
                                              C.c_void_p(s.cuda_stream))
    _check(st, "exx_energy_static")


class Plan:
    """exx_plan_create / exx_plan_destroy (the per-axis eigendecompositions, once)."""

    def __init__(self, nx, ny, nz, h, bc=(0, 0, 0), fd_order=12, omega=0.0, max_batch=64, device=0, theta=None,
                 bloch_form=0):
        lib = load_library()
        self._lib = lib
        self._h = C.c_void_p()
        self.nx, self.ny, self.nz, self.h = int(nx), int(ny), int(nz), float(h)
        self.N = self.nx * self.ny * self.nz
        self.max_batch = int(max_batch)
        self.device_index = int(device)
        self.device = torch.device("cuda", device) if device >= 0 else torch.device("cpu")
        bc_arr = (C.c_int * 3)(*[int(b) for b in bc])
        if theta is None:
            st = lib.exx_plan_create(C.byref(self._h), nx, ny, nz, h, bc_arr, fd_order, omega, max_batch, device)
            _check(st, "exx_plan_create")
        else:   # Bloch-periodic plan: theta[a] = (k-q)_a * n_a * h (exx_plan_create_bloch)
            th = (C.c_double * 3)(*[float(t) for t in theta])
            if bloch_form:      # exx_plan_create_bloch_form: the embedded complex products (cross-check form)
                st = lib.exx_plan_create_bloch_form(C.byref(self._h), nx, ny, nz, h, bc_arr, fd_order, omega, th, max_batch,
                                                    device, int(bloch_form))
            else:
                st = lib.exx_plan_create_bloch(C.byref(self._h), nx, ny, nz, h, bc_arr, fd_order, omega, th, max_batch, device)
            _check(st, "exx_plan_create_bloch")
        self._ws = None

    @classmethod
    def for_workload(cls, w, max_batch=None, device=0):
        return cls(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega,
                   max_batch if max_batch is not None else max(128, w.default_nc), device)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.exx_plan_destroy(self._h)
            self._h = C.c_void_p()
        self._ws = None
        self._aws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_variant(self, variant: int):
        _check(self._lib.exx_plan_set_variant(self._h, variant), "exx_plan_set_variant")

    def set_lanes(self, lanes: int):
        _check(self._lib.exx_plan_set_lanes(self._h, lanes), "exx_plan_set_lanes")

    def set_fusion(self, mask: int):
        """exx_plan_set_fusion: bit 0 = fused z products, bit 1 = fused x-backward + accumulate, bit 2 = half-chunk y tiles
        where nx is 8 (mod 16), bit 3 = reflection-adapted eigenbases (needs bit 0).  Default 15 = all on (exx.h)."""
        _check(self._lib.exx_plan_set_fusion(self._h, mask), "exx_plan_set_fusion")

    @property
    def fusion(self) -> int:
        return int(self._lib.exx_plan_get_fusion(self._h))

    def set_accumulate(self, on: bool):
        """exx_plan_set_accumulate: exx_apply adds into vx instead of overwriting it."""
        _check(self._lib.exx_plan_set_accumulate(self._h, 1 if on else 0), "exx_plan_set_accumulate")

    @property
    def lanes(self) -> int:
        return int(self._lib.exx_plan_get_lanes(self._h))

    def workspace_bytes(self, n_c: int = 0) -> int:
        return int(self._lib.exx_plan_workspace_bytes(self._h, n_c))

    def get_axis(self, axis: int):
        n = (self.nx, self.ny, self.nz)[axis]
        lam = np.empty(n)
        V = np.empty((n, n), order="F")  # column-major: V[i, m] = component i of eigenvector m
        _check(self._lib.exx_plan_get_axis(self._h, axis, C.c_void_p(lam.ctypes.data), C.c_void_p(V.ctypes.data)),
               "exx_plan_get_axis")
        return lam, V

    def get_axis_symmetric(self, axis: int):
        """exx_plan_get_axis_symmetric: (lam, V, n_even) of the reflection-adapted eigenbasis (even vectors first)."""
        n = (self.nx, self.ny, self.nz)[axis]
        lam = np.empty(n)
        V = np.empty((n, n), order="F")
        ne = C.c_int(0)
        _check(self._lib.exx_plan_get_axis_symmetric(self._h, axis, C.c_void_p(lam.ctypes.data), C.c_void_p(V.ctypes.data),
                                                     C.byref(ne)), "exx_plan_get_axis_symmetric")
        return lam, V, int(ne.value)

    @property
    def executed_flops_per_solve(self) -> float:
        return float(self._lib.exx_plan_executed_flops_per_solve(self._h))

    @property
    def executed_flops_per_symmetric_solve(self) -> float:
        return float(self._lib.exx_plan_executed_flops_per_symmetric_solve(self._h))

    def get_multiplier(self) -> np.ndarray:
        m = np.empty((self.nz, self.ny, self.nx))
        _check(self._lib.exx_plan_get_multiplier(self._h, C.c_void_p(m.ctypes.data)), "exx_plan_get_multiplier")
        return m

    def set_profiling(self, on: bool):
        _check(self._lib.exx_plan_set_profiling(self._h, 1 if on else 0), "exx_plan_set_profiling")

    def get_profile(self):
        """exx_plan_get_profile: {class: (ms, launches)} for classes mode_product / pair_density /
        accumulate / other, accumulated since the last call (synchronises)."""
        ms = (C.c_double * 4)()
        cnt = (C.c_longlong * 4)()
        _check(self._lib.exx_plan_get_profile(self._h, ms, cnt), "exx_plan_get_profile")
        names = ("mode_product", "pair_density", "accumulate", "other")
        return {n: (ms[i], int(cnt[i])) for i, n in enumerate(names)}

    PASS_NAMES = ("x_forward", "y_forward", "z", "z_backward", "y_backward", "x_backward", "x_backward_orbital_side")

    def get_profile_passes(self):
        """exx_plan_get_profile_passes: {pass: (ms, launches, executed flops per pair solve)} of the records the last
        get_profile() call consumed."""
        ms = (C.c_double * 8)()
        cnt = (C.c_longlong * 8)()
        fl = (C.c_double * 8)()
        _check(self._lib.exx_plan_get_profile_passes(self._h, ms, cnt, fl), "exx_plan_get_profile_passes")
        return {n: (ms[i], int(cnt[i]), fl[i]) for i, n in enumerate(self.PASS_NAMES) if cnt[i]}

    @property
    def last_launch_count(self) -> int:
        return int(self._lib.exx_plan_last_launch_count(self._h))

    @property
    def tma_launch_count(self) -> int:
        return int(self._lib.exx_plan_tma_launch_count(self._h))

    def _release_workspaces(self):
        """Drop the cached workspace.  Work queued on a non-current stream may still be using it and the caching
        allocator only knows the allocation stream, so the device is synchronised first (a rare event: only when a
        larger n_c arrives)."""
        if self._ws is not None:
            torch.cuda.synchronize(self.device)
        self._ws = None

    @staticmethod
    def _expect(t, n: int, what: str):
        if t is not None and t.numel() != n:
            raise ValueError(f"{what}: expected {n} elements, got {t.numel()}")

    def _workspace(self, n_c: int) -> torch.Tensor:
        need = self.workspace_bytes(n_c)
        if need == 0:
            raise ValueError(f"n_c={n_c} outside 1..max_batch={self.max_batch}")
        if self._ws is None or self._ws.numel() < need:
            self._release_workspaces()
            self._ws = torch.empty(need, dtype=torch.uint8, device=self.device)
        return self._ws

    def poisson_solve(self, rhs: torch.Tensor, out: torch.Tensor | None = None, n_c: int = 0,
                      stream: torch.cuda.Stream | None = None) -> torch.Tensor:
        """exx_poisson_solve: out[b] = f(L) rhs[b] (Eq. 9).  ``out`` may be ``rhs``."""
        n_rhs = rhs.shape[0] if rhs.dim() > 1 else 1
        if rhs.numel() != n_rhs * self.N:
            raise ValueError("rhs must be [n_rhs, nz, ny, nx]")
        if out is None:
            out = torch.empty_like(rhs)
        self._expect(out, n_rhs * self.N, "out")
        ws = self._workspace(n_c)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_poisson_solve(self._h, _dev_ptr(rhs, self.device, "rhs"), _dev_ptr(out, self.device, "out"),
                                         n_rhs, n_c, C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(s.cuda_stream))
        _check(st, "exx_poisson_solve")
        return out

    def poisson_solve_nonbatch(self, rhs: torch.Tensor, out: torch.Tensor | None = None,
                               stream: torch.cuda.Stream | None = None) -> torch.Tensor:
        """exx_poisson_solve_nonbatch: the per-slice algorithm of PAPER.md:74-78 (Eq. 8), one system at a time."""
        n_rhs = rhs.shape[0] if rhs.dim() > 3 else 1
        if rhs.numel() != n_rhs * self.N:
            raise ValueError("rhs must be [n_rhs, nz, ny, nx]")
        if out is None:
            out = torch.empty_like(rhs)
        self._expect(out, n_rhs * self.N, "out")
        ws = self._workspace(1)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_poisson_solve_nonbatch(self._h, _dev_ptr(rhs, self.device, "rhs"),
                                                  _dev_ptr(out, self.device, "out"), n_rhs, C.c_void_p(ws.data_ptr()),
                                                  ws.numel(), C.c_void_p(s.cuda_stream))
        _check(st, "exx_poisson_solve_nonbatch")
        return out

    def apply(self, psi: torch.Tensor, occ: torch.Tensor, tgt: torch.Tensor, occ_tgt: torch.Tensor | None = None,
              vx: torch.Tensor | None = None, n_c: int = 0, want_ex_k: bool = True,
              stream: torch.cuda.Stream | None = None):
        """exx_apply: returns (vx [n_tgt, nz, ny, nx], e_k [n_tgt] or None, E_x 0-dim tensor or None);
        all device tensors, valid once ``stream`` (default: torch's current stream) is synchronised."""
        n_occ, n_tgt = psi.shape[0], tgt.shape[0]
        if psi.numel() != n_occ * self.N or tgt.numel() != n_tgt * self.N:
            raise ValueError("psi/tgt must be [n, nz, ny, nx]")
        if vx is None:
            vx = torch.empty((n_tgt, self.nz, self.ny, self.nx), dtype=torch.float64, device=self.device)
        self._expect(occ, n_occ, "occ")
        self._expect(occ_tgt, n_tgt, "occ_tgt")
        self._expect(vx, n_tgt * self.N, "vx")
        ex = torch.empty((), dtype=torch.float64, device=self.device) if occ_tgt is not None else None
        ex_k = torch.empty(n_tgt, dtype=torch.float64, device=self.device) if want_ex_k else None
        ws = self._workspace(n_c)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_apply(self._h, _dev_ptr(psi, self.device, "psi"), _dev_ptr(occ, self.device, "occ"), n_occ,
                                 _dev_ptr(tgt, self.device, "tgt"), _dev_ptr(occ_tgt, self.device, "occ_tgt"), n_tgt,
                                 _dev_ptr(vx, self.device, "vx"), _dev_ptr(ex, self.device, "ex"),
                                 _dev_ptr(ex_k, self.device, "ex_k"), n_c, C.c_void_p(ws.data_ptr()), ws.numel(),
                                 C.c_void_p(s.cuda_stream))
        _check(st, "exx_apply")
        return vx, ex_k, ex

    def apply_symmetric(self, psi: torch.Tensor, occ: torch.Tensor, vx: torch.Tensor | None = None, n_c: int = 0,
                        want_ex_k: bool = True, stream: torch.cuda.Stream | None = None):
        """exx_apply_symmetric: targets == orbitals, only the pairs j <= k are solved.  Returns (vx, e_k, E_x)."""
        n = psi.shape[0]
        if psi.numel() != n * self.N:
            raise ValueError("psi must be [n, nz, ny, nx]")
        if vx is None:
            vx = torch.empty((n, self.nz, self.ny, self.nx), dtype=torch.float64, device=self.device)
        self._expect(occ, n, "occ")
        self._expect(vx, n * self.N, "vx")
        ex = torch.empty((), dtype=torch.float64, device=self.device)
        ex_k = torch.empty(n, dtype=torch.float64, device=self.device) if want_ex_k else None
        ws = self._workspace(n_c)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_apply_symmetric(self._h, _dev_ptr(psi, self.device, "psi"), _dev_ptr(occ, self.device, "occ"),
                                           n, _dev_ptr(vx, self.device, "vx"), _dev_ptr(ex, self.device, "ex"),
                                           _dev_ptr(ex_k, self.device, "ex_k"), n_c, C.c_void_p(ws.data_ptr()),
                                           ws.numel(), C.c_void_p(s.cuda_stream))
        _check(st, "exx_apply_symmetric")
        return vx, ex_k, ex

    @property
    def last_solve_count(self) -> int:
        return int(self._lib.exx_plan_last_solve_count(self._h))

    # ---- Bloch-periodic complex variant: complex functions are two real planes [n, 2, nz, ny, nx] --------------
    def get_axis_bloch(self, axis: int):
        n = (self.nx, self.ny, self.nz)[axis]
        lam, Vr, Vi = np.empty(n), np.empty((n, n), order="F"), np.empty((n, n), order="F")
        _check(self._lib.exx_plan_get_axis_bloch(self._h, axis, C.c_void_p(lam.ctypes.data), C.c_void_p(Vr.ctypes.data),
                                                 C.c_void_p(Vi.ctypes.data)), "exx_plan_get_axis_bloch")
        return lam, Vr + 1j * Vi

    def _workspace_bloch(self, n_c: int) -> torch.Tensor:
        need = int(self._lib.exx_plan_workspace_bytes_bloch(self._h, n_c))
        if need == 0:
            raise ValueError(f"n_c={n_c} outside 1..max_batch={self.max_batch}")
        if self._ws is None or self._ws.numel() < need:
            self._release_workspaces()
            self._ws = torch.empty(need, dtype=torch.uint8, device=self.device)
        return self._ws

    def poisson_solve_bloch(self, rhs: torch.Tensor, out: torch.Tensor | None = None, n_c: int = 0,
                            stream: torch.cuda.Stream | None = None) -> torch.Tensor:
        """exx_poisson_solve_bloch: rhs / out are [n_rhs, 2, nz, ny, nx] (real and imaginary planes)."""
        n_rhs = rhs.shape[0]
        if rhs.numel() != n_rhs * 2 * self.N:
            raise ValueError("rhs must be [n_rhs, 2, nz, ny, nx]")
        if out is None:
            out = torch.empty_like(rhs)
        ws = self._workspace_bloch(n_c)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_poisson_solve_bloch(self._h, _dev_ptr(rhs, self.device, "rhs"), _dev_ptr(out, self.device, "out"),
                                               n_rhs, n_c, C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(s.cuda_stream))
        _check(st, "exx_poisson_solve_bloch")
        return out

    def apply_bloch(self, psi: torch.Tensor, occ: torch.Tensor, tgt: torch.Tensor, vx: torch.Tensor | None = None,
                    accumulate: bool = False, want_ex_k: bool = True, n_c: int = 0,
                    stream: torch.cuda.Stream | None = None):
        """exx_apply_bloch for one (k,q) pair: psi [n_occ, 2, nz, ny, nx], tgt [n_tgt, 2, ...]; returns (vx, e_k)."""
        n_occ, n_tgt = psi.shape[0], tgt.shape[0]
        if psi.numel() != n_occ * 2 * self.N or tgt.numel() != n_tgt * 2 * self.N:
            raise ValueError("psi/tgt must be [n, 2, nz, ny, nx]")
        if vx is None:
            if accumulate:
                raise ValueError("accumulate=True needs vx")
            vx = torch.empty_like(tgt)
        self._expect(occ, n_occ, "occ")
        self._expect(vx, n_tgt * 2 * self.N, "vx")
        ex_k = torch.empty(n_tgt, dtype=torch.float64, device=self.device) if want_ex_k else None
        ws = self._workspace_bloch(n_c)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_apply_bloch(self._h, _dev_ptr(psi, self.device, "psi"), _dev_ptr(occ, self.device, "occ"), n_occ,
                                       _dev_ptr(tgt, self.device, "tgt"), n_tgt, _dev_ptr(vx, self.device, "vx"),
                                       1 if accumulate else 0, _dev_ptr(ex_k, self.device, "ex_k"), n_c,
                                       C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(s.cuda_stream))
        _check(st, "exx_apply_bloch")
        return vx, ex_k

    def ace_workspace_bytes(self, n_orb: int, n_trial: int = 0) -> int:
        return int(self._lib.exx_ace_workspace_bytes(self._h, n_orb, n_trial))

    def _ace_ws(self, n_orb: int, n_trial: int) -> torch.Tensor:
        need = self.ace_workspace_bytes(n_orb, n_trial)
        if getattr(self, "_aws", None) is None or self._aws.numel() < need:
            if getattr(self, "_aws", None) is not None:
                torch.cuda.synchronize(self.device)   # kernels queued on any stream may still use the old block
            self._aws = None
            self._aws = torch.empty(need, dtype=torch.uint8, device=self.device)
        return self._aws

    def ace_build(self, psi: torch.Tensor, w: torch.Tensor, xi: torch.Tensor | None = None, want_M: bool = True,
                  stream: torch.cuda.Stream | None = None):
        """exx_ace_build (Eqs. 17-20, 26): returns (xi [n, nz, ny, nx], M [n, n] or None,
        info int32 0-dim device tensor).  ``xi`` may be ``w`` (in place)."""
        n = psi.shape[0]
        if psi.numel() != n * self.N or w.numel() != n * self.N:
            raise ValueError("psi/w must be [n, nz, ny, nx]")
        if xi is None:
            xi = torch.empty_like(w)
        self._expect(xi, n * self.N, "xi")
        M = torch.empty((n, n), dtype=torch.float64, device=self.device) if want_M else None
        info = torch.zeros((), dtype=torch.int32, device=self.device)
        ws = self._ace_ws(n, 0)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_ace_build(self._h, _dev_ptr(psi, self.device, "psi"), _dev_ptr(w, self.device, "w"), n,
                                     _dev_ptr(xi, self.device, "xi"), _dev_ptr(M, self.device, "M"),
                                     C.c_void_p(info.data_ptr()), C.c_void_p(ws.data_ptr()), ws.numel(),
                                     C.c_void_p(s.cuda_stream))
        _check(st, "exx_ace_build")
        return xi, M, info

    def ace_apply(self, xi: torch.Tensor, phi: torch.Tensor, out: torch.Tensor | None = None,
                  stream: torch.cuda.Stream | None = None) -> torch.Tensor:
        """exx_ace_apply (Eqs. 27-29): out = -xi (h^3 xi^T phi), [m, nz, ny, nx]."""
        n, m = xi.shape[0], phi.shape[0]
        if xi.numel() != n * self.N or phi.numel() != m * self.N:
            raise ValueError("xi/phi must be [n, nz, ny, nx]")
        if out is None:
            out = torch.empty_like(phi)
        self._expect(out, m * self.N, "out")
        ws = self._ace_ws(n, m)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_ace_apply(self._h, _dev_ptr(xi, self.device, "xi"), n, _dev_ptr(phi, self.device, "phi"), m,
                                     _dev_ptr(out, self.device, "out"), C.c_void_p(ws.data_ptr()), ws.numel(),
                                     C.c_void_p(s.cuda_stream))
        _check(st, "exx_ace_apply")
        return out

    def _ace_ws_c(self, n_orb: int, n_trial: int) -> torch.Tensor:
        need = int(self._lib.exx_ace_workspace_bytes_bloch(self._h, n_orb, n_trial))
        if getattr(self, "_aws", None) is None or self._aws.numel() < need:
            if getattr(self, "_aws", None) is not None:
                torch.cuda.synchronize(self.device)
            self._aws = None
            self._aws = torch.empty(need, dtype=torch.uint8, device=self.device)
        return self._aws

    def ace_build_bloch(self, psi: torch.Tensor, w: torch.Tensor, xi: torch.Tensor | None = None, want_M: bool = True,
                        stream: torch.cuda.Stream | None = None):
        """exx_ace_build_bloch: complex orbitals [n, 2, nz, ny, nx] (real plane, imaginary plane).
        Returns (xi, M [n, n, 2] interleaved (re, im) or None, info)."""
        n = psi.shape[0]
        if psi.numel() != 2 * n * self.N or w.numel() != 2 * n * self.N:
            raise ValueError("psi/w must be [n, 2, nz, ny, nx]")
        if xi is None:
            xi = torch.empty_like(w)
        self._expect(xi, 2 * n * self.N, "xi")
        M = torch.empty((n, n, 2), dtype=torch.float64, device=self.device) if want_M else None
        info = torch.zeros((), dtype=torch.int32, device=self.device)
        ws = self._ace_ws_c(n, 0)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_ace_build_bloch(self._h, _dev_ptr(psi, self.device, "psi"), _dev_ptr(w, self.device, "w"), n,
                                           _dev_ptr(xi, self.device, "xi"), _dev_ptr(M, self.device, "M"),
                                           C.c_void_p(info.data_ptr()), C.c_void_p(ws.data_ptr()), ws.numel(),
                                           C.c_void_p(s.cuda_stream))
        _check(st, "exx_ace_build_bloch")
        return xi, M, info

    def ace_apply_bloch(self, xi: torch.Tensor, phi: torch.Tensor, out: torch.Tensor | None = None,
                        stream: torch.cuda.Stream | None = None) -> torch.Tensor:
        """exx_ace_apply_bloch: out = -xi (h^3 xi^H phi) for complex functions [m, 2, nz, ny, nx]."""
        n, m = xi.shape[0], phi.shape[0]
        if xi.numel() != 2 * n * self.N or phi.numel() != 2 * m * self.N:
            raise ValueError("xi/phi must be [n, 2, nz, ny, nx]")
        if out is None:
            out = torch.empty_like(phi)
        self._expect(out, 2 * m * self.N, "out")
        ws = self._ace_ws_c(n, m)
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        st = self._lib.exx_ace_apply_bloch(self._h, _dev_ptr(xi, self.device, "xi"), n, _dev_ptr(phi, self.device, "phi"),
                                           m, _dev_ptr(out, self.device, "out"), C.c_void_p(ws.data_ptr()), ws.numel(),
                                           C.c_void_p(s.cuda_stream))
        _check(st, "exx_ace_apply_bloch")
        return out

    def apply_host(self, psi, occ, tgt=None, tgt_start: int = -1, n_tgt: int | None = None, occ_tgt=None,
                   vx=None, n_c: int = 0):
        """exx_apply_host: HOST buffers in, HOST results out (H2D/D2H inside the call, synchronous).
        Returns (vx, e_k, E_x) as numpy arrays / float."""
        n_occ = psi.shape[0]
        if tgt is None:
            if tgt_start < 0 or n_tgt is None:
                raise ValueError("give tgt, or tgt_start and n_tgt")
        else:
            n_tgt, tgt_start = tgt.shape[0], -1
        if vx is None:
            vx = np.empty((n_tgt, self.nz, self.ny, self.nx))
        for t, n, what in ((psi, n_occ * self.N, "psi"), (occ, n_occ, "occ"), (occ_tgt, n_tgt, "occ_tgt"),
                           (vx, n_tgt * self.N, "vx"), (tgt, n_tgt * self.N, "tgt")):
            if t is not None and (t.size if isinstance(t, np.ndarray) else t.numel()) != n:
                raise ValueError(f"{what}: expected {n} elements")
        ex = np.zeros(1)
        ex_k = np.empty(n_tgt)
        st = self._lib.exx_apply_host(self._h, _host_ptr(psi, "psi"), _host_ptr(occ, "occ"), n_occ,
                                      _host_ptr(tgt, "tgt"), tgt_start, _host_ptr(occ_tgt, "occ_tgt"), n_tgt,
                                      _host_ptr(vx, "vx"), _host_ptr(ex, "ex") if occ_tgt is not None else None,
                                      _host_ptr(ex_k, "ex_k"), n_c)
        _check(st, "exx_apply_host")
        return vx, ex_k, (float(ex[0]) if occ_tgt is not None else None)
