"""Pins of the oracle's first-moment line RV (north_star's acceptance functional; stands in for the paper's
CCF + Gaussian fit)."""
from __future__ import annotations

import numpy as np

import oracle
import workloads
from helpers import line_rvs as np_line_rvs

C_CMS = 299792.458e5
LAM0, K = 5000.0, 0.01


def _gauss_rows(shifts_cms, lc=5010.0, d=0.5, sig=0.05, P=2500, norm=3.0):
    lam = LAM0 + K * np.arange(P)
    rows = [norm * (1.0 - d * np.exp(-(lam - lc * (1.0 + v / C_CMS)) ** 2 / (2 * sig * sig))) for v in shifts_cms]
    return np.array(rows)


def test_shifted_gaussian_line_returns_its_shift():
    """The first moment of a Gaussian line displaced by lc v / c is v (window +-6 sigma: truncation ~1e-8 of the shift)."""
    shifts = np.array([-300.0, -1.0, 0.0, 0.37, 25.0, 1200.0])          # cm/s
    rows = _gauss_rows(shifts)
    rv = oracle.line_rvs(rows, LAM0, K, [5010.0], [0.3], 3.0)
    np.testing.assert_allclose(rv[:, 0], shifts, rtol=1e-6, atol=1e-3)   # 0.001 cm/s: sampling of the profile


def test_symmetric_line_on_a_pixel_has_zero_rv_and_normalisation_does_not_matter():
    rows = _gauss_rows([0.0], lc=5010.0)
    assert abs(oracle.line_rvs(rows, LAM0, K, [5010.0], [0.25], 3.0)[0, 0]) < 1e-6
    a = oracle.line_rvs(rows * 7.0, LAM0, K, [5010.0], [0.25], 21.0)
    np.testing.assert_allclose(a, oracle.line_rvs(rows, LAM0, K, [5010.0], [0.25], 3.0), atol=1e-6)


def test_windows_and_edges():
    rows = _gauss_rows([10.0])
    rv = oracle.line_rvs(rows, LAM0, K, [5000.05, 5010.0, 5024.98], [0.1, 0.3, 0.1], 3.0, edge=0)
    assert np.isnan(rv[0, 0]) and np.isnan(rv[0, 2]) and abs(rv[0, 1] - 10.0) < 1e-2   # windows off the grid -> NaN
    rv2 = oracle.line_rvs(rows, LAM0, K, [5010.0], [0.3], 3.0, edge=1000)               # window inside the edge margin
    assert np.isnan(rv2[0, 0])
    flat = np.full((1, 2500), 3.0)
    assert np.isnan(oracle.line_rvs(flat, LAM0, K, [5010.0], [0.3], 3.0)[0, 0])         # no depth: undefined


def test_equals_the_numpy_functional_used_by_the_parity_tests():
    """tests/helpers.line_rvs is an independent numpy implementation of the same definition."""
    wl = workloads.make_config2(n_pix=6000, n_phases=2, grid_n=40)
    Q, D, _ = oracle.run_workload(wl)
    sw = oracle.geometry(wl)["sum_w"]
    rows = np.vstack([Q[None, :], Q[None, :] + D])
    half = 3.0 * np.maximum(wl.line_sigmas, 0.03)
    a = oracle.line_rvs(rows, wl.lambda0, wl.dlambda, wl.line_centres, half, sw, edge=64)
    b = np_line_rvs(rows, sw, wl.lambda0, wl.dlambda, wl.line_centres, wl.line_sigmas, 0, 64)
    assert np.array_equal(np.isnan(a), np.isnan(b)) and np.sum(~np.isnan(a)) > 100
    np.testing.assert_allclose(a[~np.isnan(a)], b[~np.isnan(b)], rtol=1e-9, atol=1e-6)
