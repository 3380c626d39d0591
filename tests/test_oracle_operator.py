"""Pins for the oracle's operator pieces (CPU only): FD weights, 1-D spectra, multiplier.

Each pin is something the paper/mathematics fixes independently of oracle/exx_oracle.py:
rational textbook weights (tests/golden), polynomial exactness, circulant closed-form spectrum,
the textbook sine spectrum, the numerically integrated Fourier transform of erfc(w r)/r.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import integrate

from oracle import exx_oracle as orc


def _golden_weights(golden_dir):
    out = {}
    with open(os.path.join(golden_dir, "fd_second_derivative_weights.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p = line.split()
            out[int(p[0])] = [Fraction(x) for x in p[1:]]
    return out


def test_fd_weights_match_textbook_rationals(golden_dir):
    for order, w in _golden_weights(golden_dir).items():
        got = orc.fd_weights(order, 1.0)
        ref = np.array([float(x) for x in w])
        assert np.allclose(got, ref, rtol=2e-15, atol=0), (order, got, ref)
    # h scaling
    assert np.allclose(orc.fd_weights(12, 0.25), orc.fd_weights(12, 1.0) * 16.0, rtol=1e-15)


@pytest.mark.parametrize("order", [2, 4, 6, 8, 10, 12, 14])
def test_fd_weights_exact_on_polynomials(order):
    # stencil applied to x^p at x=0 must give d2/dx2 x^p |_0 = 2 for p=2 and 0 for every other
    # p <= order+1 (odd p vanish by symmetry; even p by the order conditions)
    n0 = order // 2
    w = orc.fd_weights(order, 1.0)
    for p in range(0, order + 2):
        s = sum(w[abs(q)] * float(q) ** p for q in range(-n0, n0 + 1))
        expect = 2.0 if p == 2 else 0.0
        assert abs(s - expect) < 1e-9 * max(1.0, float(n0) ** p * abs(w[n0])), (order, p, s)
    # and must NOT be exact at p = order+2 (the stencil is of that order, not higher)
    p = order + 2
    s = sum(w[abs(q)] * float(q) ** p for q in range(-n0, n0 + 1))
    assert abs(s) > 1e-3


@pytest.mark.parametrize("n,h,order", [(16, 0.5, 12), (48, 0.25, 12), (9, 0.3, 12), (7, 1.0, 4), (60, 0.25, 12)])
def test_periodic_spectrum_closed_form(n, h, order, golden_dir):
    # circulant matrix: eigenvalues w_0 + 2 sum_q w_q cos(2 pi m q / n) (plane waves), also when the
    # stencil wraps more than once (n=9 < 13)
    K = orc.second_derivative_matrix(n, h, orc.PERIODIC, order)
    assert np.array_equal(K, K.T)
    w = [float(x) / h ** 2 for x in _golden_weights(golden_dir)[order]]
    m = np.arange(n)
    lam = w[0] + 2 * sum(w[q] * np.cos(2 * np.pi * m * q / n) for q in range(1, len(w)))
    got = np.linalg.eigvalsh(K)
    assert np.allclose(np.sort(lam), got, rtol=0, atol=2e-13 * abs(w[0]))
    # plane wave is an eigenvector
    for mm in (0, 1, n // 3):
        v = np.cos(2 * np.pi * mm * np.arange(n) / n)
        assert np.allclose(K @ v, lam[mm] * v, atol=1e-12 * abs(w[0]))
    # rows sum to zero (constants are in the null space)
    assert np.allclose(K.sum(axis=1), 0.0, atol=1e-12 * abs(w[0]))


def test_periodic_lowest_mode_converges_to_continuum():
    # 16 points, h=0.5: lam_1 = -(2 pi/8)^2 to 12th order
    K = orc.second_derivative_matrix(16, 0.5, orc.PERIODIC, 12)
    lam = np.linalg.eigvalsh(K)
    assert abs(lam[-1]) < 1e-12
    assert abs(lam[-2] + (2 * np.pi / 8.0) ** 2) < 2e-9


@pytest.mark.parametrize("n,h", [(5, 1.0), (17, 0.25), (120, 0.25)])
def test_dirichlet_order2_sine_spectrum(n, h):
    K = orc.second_derivative_matrix(n, h, orc.DIRICHLET, 2)
    m = np.arange(1, n + 1)
    lam = -(2 - 2 * np.cos(m * np.pi / (n + 1))) / h ** 2
    assert np.allclose(np.sort(lam), np.linalg.eigvalsh(K), atol=1e-12 / h ** 2)


def test_dirichlet_order12_truncated_structure(golden_dir):
    n, h = 20, 0.25
    K = orc.second_derivative_matrix(n, h, orc.DIRICHLET, 12)
    w = [float(x) / h ** 2 for x in _golden_weights(golden_dir)[12]]
    for i in range(n):
        for j in range(n):
            expect = w[abs(i - j)] if abs(i - j) <= 6 else 0.0
            assert K[i, j] == pytest.approx(expect, rel=1e-15, abs=0)
    assert np.linalg.eigvalsh(K).max() < 0  # strictly negative definite: nothing dropped (reading R3)
    K120 = orc.second_derivative_matrix(120, 0.25, orc.DIRICHLET, 12)
    assert np.linalg.eigvalsh(K120).max() < -1e-3


def test_plan_eigenpairs_are_an_eigendecomposition():
    plan = orc.make_plan(10, 9, 11, 0.3, (orc.PERIODIC, orc.DIRICHLET, orc.PERIODIC), 12, 0.106)
    for ax, n, bc in zip(range(3), (10, 9, 11), plan.bc):
        K = orc.second_derivative_matrix(n, 0.3, bc, 12)
        V, lam = plan.V[ax], plan.lam[ax]
        assert np.allclose(V.T @ V, np.eye(n), atol=1e-13)
        assert np.allclose(K @ V, V * lam[None, :], atol=1e-11)
    assert plan.mult.shape == (11, 9, 10)
    c, b, a = 3, 4, 5
    mu = -(plan.lam[0][a] + plan.lam[1][b] + plan.lam[2][c])
    assert plan.mult[c, b, a] == pytest.approx(4 * np.pi * (1 - np.exp(-mu / (4 * 0.106 ** 2))) / mu, rel=1e-13)


# ---- multiplier (Eq. 5 as read in DESIGN.md R1-R3) ------------------------------

def test_screened_kernel_is_fourier_transform_of_erfc_coulomb():
    # F[erfc(w r)/r](k) = (4 pi / k) * int_0^inf erfc(w r) sin(k r) dr; the oracle's multiplier at
    # mu = k^2 must equal it.  This pins reading R1 (the garbled exponent of Eqs. 3/5) to the physics
    # ("erfc-screened multiplier for HSE", BASELINE.json north_star).
    omega = 0.106
    for k in (0.05, 0.2, 0.7, 1.5):
        val, _ = integrate.quad(lambda r: math.erfc(omega * r) * math.sin(k * r), 0.0, 400.0, limit=4000,
                                epsabs=1e-13, epsrel=1e-12)
        ft = 4 * np.pi / k * val
        got = float(orc.kernel_multiplier(np.array(-k * k), omega, 1e-12))
        assert got == pytest.approx(ft, rel=2e-9)


def test_multiplier_limits_and_bounds():
    mu = np.logspace(-6, 3, 200)
    omega = 0.106
    m_hse = orc.kernel_multiplier(-mu, omega, 1e-12)
    m_c = orc.kernel_multiplier(-mu, 0.0, 1e-12)
    assert np.allclose(m_c, 4 * np.pi / mu, rtol=1e-15)
    assert np.all(m_hse > 0) and np.all(m_hse <= m_c * (1 + 1e-15)) and np.all(m_hse <= np.pi / omega ** 2 * (1 + 1e-15))
    assert np.all(np.diff(m_hse) < 0)                       # monotone decreasing in mu
    # omega -> 0+ (erfc(w r) -> 1) recovers the unscreened kernel; omega -> infinity screens everything
    # (SURVEY.md 8(c) A1 states these two limits the wrong way round; R1 has them right);
    # mu -> 0 gives pi / omega^2
    big = mu > 1e-2
    assert np.allclose(orc.kernel_multiplier(-mu[big], 1e-3, 1e-30), m_c[big], rtol=1e-14)
    assert np.all(orc.kernel_multiplier(-mu, 1e4, 1e-30) <= np.pi / 1e8 * (1 + 1e-12))
    assert float(orc.kernel_multiplier(np.array(-1e-14), omega, 1e-30)) == pytest.approx(np.pi / omega ** 2, rel=1e-10)
    # zero-mode rule (reading R3)
    assert float(orc.kernel_multiplier(np.array(-1e-12), 0.0, 1e-8)) == 0.0
    assert float(orc.kernel_multiplier(np.array(1e-12), 0.0, 1e-8)) == 0.0
    assert float(orc.kernel_multiplier(np.array(-1e-12), omega, 1e-8)) == pytest.approx(math.pi / 0.106 ** 2, rel=1e-14)
