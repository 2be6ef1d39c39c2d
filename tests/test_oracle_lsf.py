"""Pins of the oracle's resolution lowering (Alg. 5; reading R-LSF).

The paper says only that the final spectrum is lowered "to match the resolution provided in the configuration
file"; the reading is a Gaussian line-spread function of FWHM lambda/R.  The pins are facts about such an LSF
(closed forms, invariants), not a second copy of the oracle's loop."""
from __future__ import annotations

import math

import numpy as np

import oracle

LAM0, K, R = 5000.0, 0.01, 115000.0
SIG_INST = LAM0 / R / (2.0 * math.sqrt(2.0 * math.log(2.0)))  # Angstrom, at 5000 A


def test_flat_spectrum_is_invariant_everywhere():
    x = np.full((3, 4000), 0.7)
    np.testing.assert_allclose(oracle.lower_resolution(x, LAM0, K, R), x, rtol=1e-14)  # (sum g a) / (sum g): rounding of ~20 terms


def test_linear_spectrum_is_invariant_in_the_interior():
    """Every output pixel uses a symmetric, normalised kernel: a + b m is reproduced exactly away from the clamped ends."""
    m = np.arange(5000, dtype=np.float64)
    x = 0.3 + 2e-4 * m
    y = oracle.lower_resolution(x, LAM0, K, R)
    J = int(math.ceil(5.0 * (LAM0 + K * 5000) / R / 2.3548 / K)) + 1
    np.testing.assert_allclose(y[J:-J], x[J:-J], rtol=1e-13)
    assert y[0] > x[0] and y[-1] < x[-1]  # clamped ends pull toward the interior values


def test_gaussian_line_broadens_in_quadrature():
    """Gaussian (sigma_l) convolved with a Gaussian LSF (sigma_inst) is a Gaussian with sigma^2 = sigma_l^2 +
    sigma_inst^2 and depth scaled by sigma_l / sigma: pins the FWHM -> sigma factor and R."""
    P = 6000
    lam = LAM0 + K * np.arange(P)
    lc, d, sl = LAM0 + 30.0, 0.6, 0.05
    x = 1.0 - d * np.exp(-(lam - lc) ** 2 / (2 * sl * sl))
    y = oracle.lower_resolution(x, LAM0, K, R)
    si = lc / R / (2.0 * math.sqrt(2.0 * math.log(2.0)))
    so = math.sqrt(sl * sl + si * si)
    expect = 1.0 - d * (sl / so) * np.exp(-(lam - lc) ** 2 / (2 * so * so))
    assert np.max(np.abs(y - expect)) < 5e-6
    # a wrong factor (e.g. FWHM used as sigma) would miss by ~1e-1
    wrong = math.sqrt(sl * sl + (lc / R) ** 2)
    assert np.max(np.abs(y - (1.0 - d * (sl / wrong) * np.exp(-(lam - lc) ** 2 / (2 * wrong * wrong))))) > 1e-2


def test_impulse_response_has_unit_area_right_width_and_symmetry():
    P, m0 = 2001, 1000
    x = np.zeros(P)
    x[m0] = 1.0
    y = oracle.lower_resolution(x, LAM0, K, R)
    assert abs(y.sum() - 1.0) < 1e-5                      # normalised LSF, sigma varies by 1e-6 per pixel
    j = np.arange(P) - m0
    var_px = float((y * j * j).sum() / y.sum())
    assert abs(var_px / (SIG_INST * (LAM0 + K * m0) / LAM0 / K) ** 2 - 1.0) < 2e-3   # 5-sigma truncation: -1.6e-4
    np.testing.assert_allclose(y[m0 + 1:m0 + 9], y[m0 - 8:m0][::-1], rtol=0, atol=1e-5 * y[m0])  # symmetric up to d sigma / d lambda
    # full width at half maximum = lambda / R (linear interpolation between samples: ~1 %)
    half = y[m0] / 2
    up = np.nonzero(y[m0:] < half)[0][0]
    frac = (y[m0 + up - 1] - half) / (y[m0 + up - 1] - y[m0 + up])
    fwhm = 2.0 * (up - 1 + frac) * K
    assert abs(fwhm / ((LAM0 + K * m0) / R) - 1.0) < 0.02
    assert np.all(y[:m0 - 12] == 0.0) and np.all(y[m0 + 12:] == 0.0)  # truncated at 5 sigma ~ 9.3 px


def test_two_passes_compose_in_quadrature():
    """LSF(R1) then LSF(R2) == LSF(R_eff), 1/R_eff^2 = 1/R1^2 + 1/R2^2 (Gaussian * Gaussian), up to truncation."""
    rng = np.random.default_rng(3)
    P = 3000
    lam = LAM0 + K * np.arange(P)
    x = 1.0 - sum(dd * np.exp(-(lam - c) ** 2 / (2 * s * s))
                  for dd, c, s in zip(rng.uniform(0.1, 0.8, 12), rng.uniform(LAM0 + 2, LAM0 + 28, 12), rng.uniform(0.02, 0.08, 12)))
    R1, R2 = 150000.0, 180000.0
    Re = 1.0 / math.sqrt(1 / R1 ** 2 + 1 / R2 ** 2)
    two = oracle.lower_resolution(oracle.lower_resolution(x, LAM0, K, R1), LAM0, K, R2)
    one = oracle.lower_resolution(x, LAM0, K, Re)
    assert np.max(np.abs(two - one)[50:-50]) < 2e-5


def test_infinite_resolution_and_switch_off():
    rng = np.random.default_rng(4)
    x = rng.uniform(0.2, 1.0, (2, 800))
    np.testing.assert_allclose(oracle.lower_resolution(x, LAM0, K, 1e12), x, rtol=1e-15)
    np.testing.assert_array_equal(oracle.lower_resolution(x, LAM0, K, 0.0), x)


def test_rows_are_independent_and_the_operator_is_linear():
    rng = np.random.default_rng(5)
    a, b = rng.uniform(0, 1, (2, 1500))
    both = oracle.lower_resolution(np.stack([a, b]), LAM0, K, R)
    np.testing.assert_array_equal(both[0], oracle.lower_resolution(a, LAM0, K, R))
    np.testing.assert_allclose(oracle.lower_resolution(2 * a - 3 * b, LAM0, K, R), 2 * both[0] - 3 * both[1], atol=1e-14)
