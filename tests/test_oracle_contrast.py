"""Pins of the oracle's SOAPcontrast: the per-pixel ratio of two Planck functions.

The function is a closed form, so it is pinned by what physics and arithmetic fix independently of its own
formula: the equal-temperature identity, the Wien and Rayleigh-Jeans limits, a value worked out by hand at the
wavelength and temperatures the paper quotes for SOAP 2.0's fixed contrast (5293 A, 5778 K, spot 663 K cooler;
P:300 and its footnote 4), Wien's displacement law recovered from the function, and the chromatic trend the
paper states ("the absolute value of the contrast in the blue part of the spectrum is higher than in the
red part").  Not a GPU test.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

import oracle

# CODATA 2018 exact SI values, typed here independently of the oracle's own defines
H, C, KB = 6.62607015e-34, 299792458.0, 1.380649e-23


def test_equal_temperatures_give_one():
    c = oracle.contrast_planck(3800.0, 0.01, 5000, 5778.0, 5778.0)
    assert np.all(c == 1.0)


def test_hand_value_at_the_papers_reference_wavelength():
    """5293 A, quiet 5778 K, spot 5778 - 663 = 5115 K (footnote 4), worked out step by step:
    h c / k_B = 1.438776877e-2 m K;  x_q = 1.438776877e-2 / (5.293e-7 * 5778) = 4.704527...;
    x_a = 1.438776877e-2 / (5.293e-7 * 5115) = 5.314317...;  (e^x_q - 1) / (e^x_a - 1) = 0.54119..."""
    hc_k = H * C / KB
    assert abs(hc_k - 1.438776877e-2) < 1e-11
    xq = hc_k / (5.293e-7 * 5778.0)
    xa = hc_k / (5.293e-7 * 5115.0)
    assert abs(xq - 4.7045) < 5e-4 and abs(xa - 5.3143) < 5e-4
    hand = (math.exp(xq) - 1.0) / (math.exp(xa) - 1.0)
    assert abs(hand - 0.5412) < 5e-4
    got = oracle.contrast_planck(5293.0, 0.01, 1, 5778.0, 5115.0)[0]
    assert abs(got / hand - 1.0) < 1e-13


def test_wien_limit():
    """x >> 1 (short wavelength): the -1 terms vanish and the ratio tends to exp(-(hc / lambda k)(1/T_a - 1/T_q))."""
    lam0, k, n = 500.0, 0.5, 200   # 500-600 A: x ~ 40-60
    tq, ta = 5778.0, 4700.0
    got = oracle.contrast_planck(lam0, k, n, tq, ta)
    lam = (lam0 + k * np.arange(n)) * 1e-10
    wien = np.exp(-(H * C / (lam * KB)) * (1.0 / ta - 1.0 / tq))
    assert np.max(np.abs(got / wien - 1.0)) < 1e-12


def test_rayleigh_jeans_limit():
    """x << 1 (long wavelength): B_lambda ~ 2 c k T / lambda^4, so the ratio tends to T_a / T_q, from below for a cool
    region, with the first-order correction (1 + x_q / 2) / (1 + x_a / 2)."""
    tq, ta = 5778.0, 4700.0
    got = oracle.contrast_planck(1e9, 1e8, 5, tq, ta)   # 10-14 cm
    lam = (1e9 + 1e8 * np.arange(5)) * 1e-10
    xq, xa = H * C / (lam * KB * tq), H * C / (lam * KB * ta)
    assert np.all(got < ta / tq) and np.max(np.abs(got / (ta / tq) - 1.0)) < 5e-5
    assert np.max(np.abs(got / ((ta / tq) * (1 + xq / 2) / (1 + xa / 2)) - 1.0)) < 1e-9


def test_monotonic_and_chromatic():
    """A cool spot is darker everywhere and darker in the blue than in the red; a hot facula the reverse."""
    spot = oracle.contrast_planck(3800.0, 1.0, 3101, 5778.0, 4700.0)
    assert np.all(spot < 1.0) and np.all(np.diff(spot) > 0.0)
    assert spot[0] < 0.25 < spot[-1]         # 3800 A: 0.205; 6900 A: 0.433
    fac = oracle.contrast_planck(3800.0, 1.0, 3101, 5778.0, 6000.0)
    assert np.all(fac > 1.0) and np.all(np.diff(fac) < 0.0)
    # swapping the two temperatures inverts the ratio
    inv = oracle.contrast_planck(3800.0, 1.0, 3101, 4700.0, 5778.0)
    assert np.max(np.abs(spot * inv - 1.0)) < 1e-14


def test_reconstructs_wiens_displacement_law():
    """B_lambda(T) itself, rebuilt from the ratio against a fixed reference temperature, peaks at lambda T = 2.897771955e-3 m K.
    (ratio * B_ref, with B_ref typed here in its textbook form: only the ratio comes from the oracle.)"""
    t_ref, t = 5000.0, 5778.0
    lam0, k, n = 3000.0, 0.5, 10001           # 3000-8000 A
    ratio = oracle.contrast_planck(lam0, k, n, t_ref, t)
    lam = (lam0 + k * np.arange(n)) * 1e-10
    b_ref = 2 * H * C * C / lam ** 5 / np.expm1(H * C / (lam * KB * t_ref))
    peak = lam[np.argmax(ratio * b_ref)]
    assert abs(peak * t / 2.897771955e-3 - 1.0) < 2e-4   # half a grid step of 0.5 A at 5015 A is 1e-4


def test_matches_the_input_generator_used_by_the_workloads():
    """workloads.synth.planck_ratio (input preparation, numpy) is an independent typing of the same ratio."""
    from workloads.synth import planck_ratio
    lam = 3800.0 + 0.01 * np.arange(310000)
    a = planck_ratio(lam, 4700.0, 5778.0)
    b = oracle.contrast_planck(3800.0, 0.01, 310000, 5778.0, 4700.0)
    assert np.max(np.abs(a / b - 1.0)) < 1e-9   # the generator's h c / k_B constant is typed to 10 digits


def test_bad_arguments():
    with pytest.raises(RuntimeError):
        oracle.contrast_planck(5000.0, 0.01, 10, 0.0, 4700.0)
    with pytest.raises(RuntimeError):
        oracle.contrast_planck(5000.0, 0.01, 10, 5778.0, -1.0)
