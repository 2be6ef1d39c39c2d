"""Pins of the oracle's flux-only / CB-only outputs (Eq. 1-2).

None of these retypes the oracle's formula: each is a closed form, an invariant, a library routine
(numpy.interp in the twin) or a brute-force enumeration by hand."""
from __future__ import annotations

import math

import numpy as np
import pytest

import oracle
from oracle import soap_oracle_np as onp
import workloads

TOTAL, FLUX, CB = 0, 1, 2
C_KMS = 299792.458


def _wl():
    wl = workloads.make_config3(n_pix=700, n_phases=5, grid_n=36)
    wl.vsini_kms = 9.0
    wl.incl_deg = 70.0
    wl.regions = [(-10.0, 160.0, 0.3, 2), (15.0, 190.0, 0.2, 1)]
    wl.phases = np.array([0.0, 0.05, 0.1, 0.5, 0.95])
    return wl


def _run(wl, effect, **kw):
    args = dict(C_spot=wl.spot_contrast, C_facula=wl.facula_contrast, lb_spot=wl.spot_lb, lb_facula=wl.facula_lb)
    args.update(kw)
    return oracle.active(wl, wl.quiet, wl.spot, wl.facula, wl.lambda0, wl.dlambda, wl.regions, wl.phases,
                         effect=effect, **args)


def test_effects_equal_numpy_twin():
    wl = _wl()
    cells = onp.geometry(wl.grid_n, wl.vsini_kms, wl.incl_deg, wl.ld_u1, wl.ld_u2, wl.mu_centres)
    for effect in (TOTAL, FLUX, CB):
        D, na = _run(wl, effect)
        Dn, nan = onp.active(cells, wl.incl_deg, wl.quiet, wl.spot, wl.facula, wl.spot_contrast, wl.facula_contrast,
                             wl.spot_lb, wl.facula_lb, wl.lambda0, wl.dlambda, wl.regions, wl.phases, effect=effect)
        assert list(na) == list(nan) and max(na) > 0
        np.testing.assert_allclose(D, Dn, rtol=0, atol=1e-10 * np.max(np.abs(Dn)))


def test_unit_intensity_ratio_kills_the_flux_effect_and_cb_equals_total():
    """I_ratio == 1 (no contrast array, LB == 1): Eq. 1 vanishes identically and Eq. 2 == Eq. 3."""
    wl = _wl()
    kw = dict(C_spot=None, C_facula=None, lb_spot=(1.0, 0.0, 0.0), lb_facula=(1.0, 0.0, 0.0))
    Df, _ = _run(wl, FLUX, **kw)
    Dc, _ = _run(wl, CB, **kw)
    Dt, _ = _run(wl, TOTAL, **kw)
    assert np.all(Df == 0.0)
    assert np.max(np.abs(Dt)) > 0
    np.testing.assert_array_equal(Dc, Dt)


def test_identical_spectra_kill_the_cb_effect_and_flux_equals_total():
    """S_active == S_quiet: Eq. 2 vanishes identically and Eq. 1 == Eq. 3."""
    wl = _wl()
    wl.spot = wl.quiet.copy()
    wl.facula = wl.quiet.copy()
    Dc, _ = _run(wl, CB)
    Df, _ = _run(wl, FLUX)
    Dt, _ = _run(wl, TOTAL)
    assert np.all(Dc == 0.0)
    np.testing.assert_array_equal(Df, Dt)
    assert np.max(np.abs(Dt)) > 0


def test_flux_effect_of_a_flat_continuum_is_closed_form():
    """S_quiet == a, constant contrast c, LB(mu) = l0 + l1 mu:  Delta_flux = a * sum_covered w (c LB(mu) - 1) at
    every pixel (the shift of a constant is the constant, reading S8), whatever the active spectrum is."""
    wl = _wl()
    a, c = 0.75, 0.55  # a is exact in the fp32 input table
    wl.quiet = np.full_like(wl.quiet, a)
    wl.regions = [(15.0, 190.0, 0.25, 1)]
    lb = (0.9, 0.2, 0.0)
    D, na = _run(wl, FLUX, C_spot=np.full(wl.n_pix, c), lb_spot=lb)
    g = oracle.geometry(wl)
    for p, ph in enumerate(wl.phases):
        tm, n = oracle.info_map(wl, wl.regions, ph)
        cov = tm == 1
        expect = a * float(np.sum(g["w"][cov] * (c * (lb[0] + lb[1] * g["mu"][cov]) - 1.0)))
        assert n == na[p]
        np.testing.assert_allclose(D[p], expect, rtol=1e-11, atol=1e-12)
    assert max(na) > 0


def test_effects_decompose_the_total():
    """Eq. 3 = Eq. 1 + Eq. 2 + the cross term sum w (I_ratio - 1)(S'_active - S'_quiet).  With a constant intensity
    ratio r (flat contrast, LB == 1) the cross term is (r - 1) * Delta_cb, so total = flux + r * cb."""
    wl = _wl()
    r = 0.6
    kw = dict(C_spot=np.full(wl.n_pix, r), C_facula=np.full(wl.n_pix, r), lb_spot=(1.0, 0.0, 0.0), lb_facula=(1.0, 0.0, 0.0))
    Dt, _ = _run(wl, TOTAL, **kw)
    Df, _ = _run(wl, FLUX, **kw)
    Dc, _ = _run(wl, CB, **kw)
    np.testing.assert_allclose(Dt, Df + r * Dc, rtol=0, atol=1e-12 * np.max(np.abs(Dt)))


def test_effects_by_hand_on_the_5x5_grid():
    """Brute force: region (lat 0, lon 0, radius 0.5, i = 90, phase 0) covers the centre cell and its 4 edge
    neighbours of the 5x5 grid (pin P6, tests/golden/grid5_by_hand.txt); each effect enumerated cell by cell with
    an explicit search-based interpolation."""
    st = dict(grid_n=5, vsini_kms=30.0, incl_deg=90.0, ld_u1=0.29, ld_u2=0.34, mu_centres=np.array([1.0]), doppler_mode=0)
    from types import SimpleNamespace
    st = SimpleNamespace(**st)
    P, lam0, k = 300, 5000.0, 0.02
    lam = [lam0 + k * m for m in range(P)]
    rng = np.random.default_rng(11)
    Sq = rng.uniform(0.3, 1.0, P)
    Ss = rng.uniform(0.3, 1.0, P)
    C = rng.uniform(0.4, 0.7, P)
    lb = (0.8, 0.3, 0.1)
    covered = [(0.0, 0.0), (0.4, 0.0), (-0.4, 0.0), (0.0, 0.4), (0.0, -0.4)]

    def lerp(S, x):
        if x <= lam[0]:
            return S[0]
        if x >= lam[-1]:
            return S[-1]
        n = 0
        while lam[n + 1] < x:
            n += 1
        t = (x - lam[n]) / (lam[n + 1] - lam[n])
        return S[n] + t * (S[n + 1] - S[n])

    expect = {e: np.zeros(P) for e in (TOTAL, FLUX, CB)}
    for x, y in covered:
        mu = math.sqrt(1 - x * x - y * y)
        w = 1 - 0.29 * (1 - mu) - 0.34 * (1 - mu) ** 2
        beta = x * 30.0 / C_KMS
        Dop = math.sqrt((1 - beta) / (1 + beta))
        LB = lb[0] + lb[1] * mu + lb[2] * mu * mu
        for m in range(P):
            sq, sa = lerp(Sq, lam[m] * Dop), lerp(Ss, lam[m] * Dop)
            I = C[m] * LB
            expect[TOTAL][m] += w * (I * sa - sq)
            expect[FLUX][m] += w * (I * sq - sq)
            expect[CB][m] += w * (sa - sq)
    for e in (TOTAL, FLUX, CB):
        D, na = oracle.active(st, Sq[None, :], Ss[None, :], None, lam0, k, [(0.0, 0.0, 0.5, 1)], np.array([0.0]),
                              C_spot=C, lb_spot=lb, effect=e)
        assert list(na) == [5]
        np.testing.assert_allclose(D[0], expect[e], rtol=0, atol=2e-10)


def test_unknown_effect_is_rejected():
    wl = _wl()
    with pytest.raises(RuntimeError):
        _run(wl, 3)
