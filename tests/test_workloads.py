"""Input generators: determinism, orthonormality under h^3, occupations, config table (CPU only)."""
import json
import os

import numpy as np
import torch

from paper_2501_16572_b200 import workloads as wl


def test_config_table_matches_baseline_json():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cfgs = json.load(open(os.path.join(root, "BASELINE.json")))["configs"]
    assert len(cfgs) == len(wl.WORKLOADS) == 5
    expect = {1: (16, 16, 16, 64), 2: (48, 48, 48, 4096), 3: (60, 60, 120, 65536),
              4: (96, 96, 96, 393216), 5: (120, 120, 120, 409600)}
    for i, w in wl.WORKLOADS.items():
        assert (w.nx, w.ny, w.nz, w.pair_solves) == expect[i]
        assert f"{w.nx}x{w.ny}x{w.nz}" in cfgs[i - 1].replace(" ", "")
        assert w.order == 12
    assert wl.WORKLOADS[3].bc == (wl.PERIODIC, wl.PERIODIC, wl.DIRICHLET)
    assert wl.WORKLOADS[1].omega <= 0 and wl.WORKLOADS[2].omega == 0.106


def test_orbitals_are_seeded_and_orthonormal():
    w = wl.WORKLOADS[1]
    a = wl.make_orbitals(w)
    b = wl.make_orbitals(w)
    assert torch.equal(a, b)
    assert a.shape == (8, 16, 16, 16) and a.dtype == torch.float64
    G = (a.view(8, -1) @ a.view(8, -1).T) * w.h ** 3
    assert torch.allclose(G, torch.eye(8, dtype=torch.float64), atol=1e-13)


def test_smoothed_slab_orbitals():
    w = wl.scaled(wl.WORKLOADS[3], 6)
    psi, occ, tgt, occ_t = wl.make_inputs(w)
    assert psi.shape == (6, 120, 60, 60) and tgt.shape[0] == 6
    G = (psi.view(6, -1) @ psi.view(6, -1).T) * w.h ** 3
    assert torch.allclose(G, torch.eye(6, dtype=torch.float64), atol=1e-12)
    # confined by the envelope: the first/last z planes carry little weight
    zprof = (psi ** 2).sum(dim=(0, 2, 3))
    assert zprof[0] < 0.05 * zprof.max() and zprof[-1] < 0.05 * zprof.max()  # exp(-(14.9/8)^2) ~ 0.03
    # smoothing: neighbouring points are strongly correlated
    x = psi[0]
    c = (x[:, :, 1:] * x[:, :, :-1]).sum() / (x * x).sum()
    assert c > 0.8


def test_fermi_dirac_occupations():
    w = wl.WORKLOADS[3]
    occ = wl.occupations(w)
    assert occ.shape == (256,) and np.all(np.diff(occ) <= 0) and occ[0] > 2 - 1e-12 and 0 < occ[-1] < 1e-12
    i_mu = int(round(0.7 * 255))
    assert abs(occ[i_mu] - 1.0) < 0.2
    assert np.all(wl.occupations(wl.WORKLOADS[2]) == 2.0)
    w4 = wl.WORKLOADS[4]
    o4 = wl.occupations(w4)[w4.tgt_start:w4.tgt_start + w4.n_tgt]
    assert o4[0] > 1.99 and o4[-1] < 0.02     # the target block straddles the Fermi edge
