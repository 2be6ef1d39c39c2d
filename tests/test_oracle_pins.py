"""Pins P1-P10 of DESIGN.md section 4: the fp64 oracle checked against things other than itself.

Each test says which plausible oracle mistake it would catch.  All CPU-only (-m "not gpu").
"""
from __future__ import annotations

import bisect
import math
import os
from types import SimpleNamespace

import numpy as np
import pytest

import oracle
from oracle import soap_oracle_np as onp
import workloads

C_KMS = 299792.458
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def star(N=50, vsini=2.0, incl=90.0, u1=0.29, u2=0.34, mu_centres=(1.0,), mode=0):
    return SimpleNamespace(grid_n=N, vsini_kms=vsini, incl_deg=incl, ld_u1=u1, ld_u2=u2,
                           mu_centres=np.asarray(mu_centres, dtype=np.float64), doppler_mode=mode)


def gaussian_spectrum(P, lambda0, k, centres, depths, sigmas):
    lam = lambda0 + k * np.arange(P)
    S = np.ones(P)
    for c, d, s in zip(centres, depths, sigmas):
        S -= d * np.exp(-0.5 * ((lam - c) / s) ** 2)
    return S


MU20 = 0.05 * (np.arange(20) + 1.0)


# ------------------------------------------------------------------------------------------------
# P1: v sin i = 0, no limb darkening  =>  Q = S * n_visible at every pixel
#     catches: any shift applied at v = 0, a weight that is not exactly 1, wrong visible count
# ------------------------------------------------------------------------------------------------
def test_p1_identity_at_zero_rotation():
    st = star(N=40, vsini=0.0, u1=0.0, u2=0.0)
    S = gaussian_spectrum(3000, 5000.0, 0.01, [5010.0, 5017.3], [0.5, 0.3], [0.05, 0.04])
    Q = oracle.quiet(st, S[None, :], 5000.0, 0.01)
    g = oracle.geometry(st)
    # number of cell centres inside the unit circle, counted independently
    xs = -1.0 + (2.0 * np.arange(40) + 1.0) / 40
    n_vis = int(np.sum(xs[:, None] ** 2 + xs[None, :] ** 2 <= 1.0))
    assert g["n_visible"] == n_vis
    # (lam_m - lam_0)/k is m only to within an ulp, so the closed-form index may land an ulp below m:
    # the lerp then returns S[m] to ~1e-12 relative instead of exactly
    np.testing.assert_allclose(Q, S * n_vis, rtol=2e-11, atol=0)


# ------------------------------------------------------------------------------------------------
# P2: flat continuum is invariant under shifting  =>  Q = a * sum_w at EVERY pixel (needs the clamp)
#     catches: edge handling that reads zeros / garbage outside the grid, weight errors
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0, 1])
def test_p2_flat_continuum(mode):
    st = star(N=30, vsini=20.0, mu_centres=MU20, mode=mode)
    S = np.full((20, 500), 0.73)
    Q = oracle.quiet(st, S, 6000.0, 0.01)
    g = oracle.geometry(st)
    np.testing.assert_allclose(Q, 0.73 * g["sum_w"], rtol=1e-13)


# ------------------------------------------------------------------------------------------------
# P3: linear interpolation reproduces linear functions: S = a + b lam
#     => Q[m] = a sum_w + b lam_m sum_c w_c D_c   in the interior.  Checks D and w jointly,
#     with D and w recomputed here from their definitions.
#     catches: wrong Doppler factor / sign, inverted gather (D vs 1/D), wrong LD law, transposed x/y
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [0, 1])
def test_p3_linear_spectrum_closed_form(mode):
    N, vsini, incl, u1, u2 = 24, 15.0, 70.0, 0.4, 0.2
    st = star(N=N, vsini=vsini, incl=incl, u1=u1, u2=u2, mode=mode)
    P, lam0, k = 4000, 5000.0, 0.01
    lam = lam0 + k * np.arange(P)
    a, b = 2.0, 3e-4
    Q = oracle.quiet(st, (a + b * lam)[None, :], lam0, k)
    sw = 0.0
    swd = 0.0
    for j in range(N):
        for i in range(N):
            x = -1 + (2 * j + 1) / N
            y = -1 + (2 * i + 1) / N
            if x * x + y * y > 1:
                continue
            mu = math.sqrt(1 - x * x - y * y)
            w = 1 - u1 * (1 - mu) - u2 * (1 - mu) ** 2
            beta = x * vsini * math.sin(math.radians(incl)) / C_KMS
            # receding (+x) cells are red-shifted: the light seen at lam left the star at lam / (1+z)
            D = math.sqrt((1 - beta) / (1 + beta)) if mode == 0 else 1 - beta
            sw += w
            swd += w * D
    inner = slice(50, P - 50)
    np.testing.assert_allclose(Q[inner], a * sw + b * lam[inner] * swd, rtol=2e-13)


def test_doppler_sign_receding_limb_is_redshifted():
    """Sign pin: +x is the receding limb (v > 0) and a receding cell's line moves to LONGER wavelength
    by lambda * sqrt((1+beta)/(1-beta)) (Eq. 6).  catches: flipped velocity sign, D inverted."""
    st = star(N=10, vsini=50.0)
    g = oracle.geometry(st)
    N = 10
    c = 9 * N + 5  # j = 9 (x = +0.9), i = 5
    assert g["visible"][c] and g["vel"][c] > 0 and g["x"][c] > 0
    assert g["D"][c] < 1.0
    P, lam0, k = 6000, 5000.0, 0.005
    lam = lam0 + k * np.arange(P)
    lc, sig = 5015.0, 0.04
    S = 1 - 0.5 * np.exp(-0.5 * ((lam - lc) / sig) ** 2)
    out = oracle.shifted_row(S, lam0, k, g["D"][c])
    centroid = np.sum(lam * (1 - out)) / np.sum(1 - out)
    beta = g["vel"][c] / C_KMS
    expect = lc * math.sqrt((1 + beta) / (1 - beta))
    assert expect > lc
    assert abs(centroid - expect) < 2e-6


# ------------------------------------------------------------------------------------------------
# P4: Gaussian line, linear limb darkening, solid-body rotation  ==  analytic rotational broadening
#     (Gray, "Observation and Analysis of Stellar Photospheres", G(x) ~ 2(1-eps) sqrt(1-x^2) +
#     (pi eps / 2)(1 - x^2)) convolved with the Gaussian, within grid-convergence error.
#     catches: wrong velocity field (v not proportional to x), wrong LD weighting, missing cells
# ------------------------------------------------------------------------------------------------
def _rot_broadened_gaussian(lam, lc, d, sigma, eps, vsini):
    dl = lc * vsini / C_KMS
    n = 4001
    th = np.linspace(-np.pi / 2, np.pi / 2, n)
    x = np.sin(th)
    G = (2 * (1 - eps) * np.sqrt(np.maximum(0, 1 - x * x)) + 0.5 * np.pi * eps * (1 - x * x)) / (
        np.pi * (1 - eps / 3))  # integrates to 1 over x in [-1,1]
    wts = G * np.cos(th)
    wts[0] *= 0.5
    wts[-1] *= 0.5
    wts *= th[1] - th[0]
    assert abs(wts.sum() - 1) < 1e-6
    prof = np.exp(-0.5 * ((lam[:, None] - lc - x[None, :] * dl) / sigma) ** 2) @ wts
    return 1 - d * prof


@pytest.mark.parametrize("N,tol", [(100, 4e-5), (200, 2e-5), (300, 1e-5)])
def test_p4_rotational_broadening_kernel(N, tol):
    eps, vsini, d, sigma, k = 0.6, 2.0, 0.6, 0.05, 0.01
    P, lam0 = 1200, 5000.0
    lc = lam0 + k * 600
    lam = lam0 + k * np.arange(P)
    S = 1 - d * np.exp(-0.5 * ((lam - lc) / sigma) ** 2)
    st = star(N=N, vsini=vsini, u1=eps, u2=0.0)
    Q = oracle.quiet(st, S[None, :], lam0, k)
    f = Q / oracle.geometry(st)["sum_w"]
    # linear interpolation with uniformly spread sub-pixel offsets == smoothing by a triangular kernel
    # of variance k^2/6: fold that into sigma (depth rescaled to conserve equivalent width)
    sig_eff = math.sqrt(sigma ** 2 + k * k / 6)
    model = _rot_broadened_gaussian(lam, lc, d * sigma / sig_eff, sig_eff, eps, vsini)
    res = np.max(np.abs(f - model)[100:-100])
    assert res < tol, res
    # and without the correction the residual is the (larger) interpolation-smoothing floor, still small
    raw = np.max(np.abs(f - _rot_broadened_gaussian(lam, lc, d, sigma, eps, vsini))[100:-100])
    assert res < raw < 5e-3


def test_p4_residual_decreases_with_grid():
    eps, vsini, d, sigma, k = 0.6, 2.0, 0.6, 0.05, 0.01
    P, lam0 = 1200, 5000.0
    lc = lam0 + k * 600
    lam = lam0 + k * np.arange(P)
    S = 1 - d * np.exp(-0.5 * ((lam - lc) / sigma) ** 2)
    sig_eff = math.sqrt(sigma ** 2 + k * k / 6)
    model = _rot_broadened_gaussian(lam, lc, d * sigma / sig_eff, sig_eff, eps, vsini)
    res = []
    for N in (50, 100, 200, 300):
        st = star(N=N, vsini=vsini, u1=eps, u2=0.0)
        f = oracle.quiet(st, S[None, :], lam0, k) / oracle.geometry(st)["sum_w"]
        res.append(np.max(np.abs(f - model)[100:-100]))
    assert res[0] > res[1] > res[2] > res[3]


# ------------------------------------------------------------------------------------------------
# P5: mirror symmetry: a region at effective longitude +L and -L gives wavelength-mirrored deltas
#     catches: asymmetric membership test, phase sign / origin errors, x <-> -x slips in velocity
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("incl", [90.0, 60.0])
def test_p5_mirror_symmetry(incl):
    N, P, lam0, k = 60, 2001, 5000.0, 0.01
    lc = lam0 + k * 1000  # exactly on a pixel
    lam = lam0 + k * np.arange(P)
    row = 1 - 0.6 * np.exp(-0.5 * ((lam - lc) / 0.05) ** 2)
    Sq = np.tile(row, (20, 1))                   # identical rows in every mu bin
    Ss = 0.5 * np.tile(1 - 0.66 * np.exp(-0.5 * ((lam - lc) / 0.05) ** 2), (20, 1))
    st = star(N=N, vsini=2.0, incl=incl, mu_centres=MU20)
    regions = [(25.0, 180.0, 0.2, 1)]
    ph = np.array([0.5 - 0.11, 0.5 + 0.11])      # effective longitude -39.6 deg and +39.6 deg
    D, na = oracle.active(st, Sq, Ss, None, lam0, k, regions, ph)
    assert na[0] == na[1] > 0
    scale = np.max(np.abs(D))
    inner = slice(200, P - 200)
    mirrored = D[1][::-1]
    assert np.max(np.abs(D[0] - mirrored)[inner]) <= 1e-5 * scale
    # and the two are genuinely different spectra (the test is not vacuous)
    assert np.max(np.abs(D[0] - D[1])[inner]) > 1e-2 * scale


# ------------------------------------------------------------------------------------------------
# P6: 5x5 grid by hand / brute force with an independent interpolation (search, not closed form)
#     catches: index slips (j/i swap, off-by-one), wrong cell centres, wrong visibility rule, wrong w
# ------------------------------------------------------------------------------------------------
def _golden5():
    vals = {"mu": [], "w": []}
    with open(os.path.join(GOLDEN, "grid5_by_hand.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            key, *rest = line.split()
            if key == "mu":
                vals["mu"].append((float(rest[0]), int(rest[1])))
            elif key == "w":
                vals["w"].append(float(rest[0]))
            elif key in ("n_visible",):
                vals[key] = int(rest[0])
            elif key == "sum_w":
                vals[key] = float(rest[0])
            else:
                vals[key] = sorted(tuple(float(v) for v in tok.split(",")) for tok in rest)
    return vals


def _lerp_by_search(lam, S, x):
    """Linear interpolation by bracketing search on the actual wavelength array (no closed-form index)."""
    if x <= lam[0]:
        return S[0]
    if x >= lam[-1]:
        return S[-1]
    n = bisect.bisect_right(lam, x) - 1
    return S[n] + (S[n + 1] - S[n]) * (x - lam[n]) / (lam[n + 1] - lam[n])


def test_p6_grid5_by_hand():
    gold = _golden5()
    st = star(N=5, vsini=30.0, u1=0.29, u2=0.34)
    g = oracle.geometry(st)
    assert g["n_visible"] == gold["n_visible"] == 21
    assert abs(g["sum_w"] - gold["sum_w"]) < 5e-7
    mus = np.sort(g["mu"][g["visible"] == 1])[::-1]
    expect = np.sort(np.concatenate([[m] * n for m, n in gold["mu"]]))[::-1]
    np.testing.assert_allclose(mus, expect, atol=5e-7)
    ws = np.sort(np.unique(np.round(g["w"][g["visible"] == 1], 6)))[::-1]
    np.testing.assert_allclose(ws, gold["w"], atol=1e-6)
    # exact forms: r^2 in {0, .16, .32, .64, .80}
    for r2, n in [(0.0, 1), (0.16, 4), (0.32, 4), (0.64, 4), (0.80, 8)]:
        assert int(np.sum(np.isclose(g["mu"][g["visible"] == 1], math.sqrt(1 - r2), atol=1e-12))) == n
    # only 5 distinct velocities x * vsini
    v = np.unique(np.round(g["vel"][g["visible"] == 1], 9))
    np.testing.assert_allclose(v, 30.0 * np.array([-0.8, -0.4, 0.0, 0.4, 0.8]), atol=1e-9)

    # brute force the integrated spectrum by explicit enumeration of the 21 cells
    P, lam0, k = 400, 5000.0, 0.02
    lam = [lam0 + k * m for m in range(P)]
    rng = np.random.default_rng(5)
    S = rng.uniform(0.2, 1.0, P)
    Q = oracle.quiet(st, S[None, :], lam0, k)
    coords = [-0.8, -0.4, 0.0, 0.4, 0.8]
    Qb = np.zeros(P)
    for x in coords:
        for y in coords:
            if x * x + y * y > 1.0:
                continue
            mu = math.sqrt(1 - x * x - y * y)
            w = 1 - 0.29 * (1 - mu) - 0.34 * (1 - mu) ** 2
            beta = x * 30.0 / C_KMS
            D = math.sqrt((1 - beta) / (1 + beta))
            for m in range(P):
                Qb[m] += w * _lerp_by_search(lam, S, lam[m] * D)
    # a white-noise spectrum turns the ~5e-11 px rounding of the source coordinate into ~1e-11 relative
    np.testing.assert_allclose(Q, Qb, rtol=2e-10)


def test_p6_grid5_region_membership():
    gold = _golden5()
    st = star(N=5)
    coords = np.array([-0.8, -0.4, 0.0, 0.4, 0.8])
    for phase, key in [(0.0, "active_phase0"), (0.125, "active_phase0125")]:
        tm, n = oracle.info_map(st, [(0.0, 0.0, 0.5, 1)], phase)
        got = sorted((float(coords[c // 5]), float(coords[c % 5])) for c in np.flatnonzero(tm))
        assert got == gold[key], (phase, got)
        assert n == len(gold[key])


# ------------------------------------------------------------------------------------------------
# P7: sum of weights -> N^2 (pi/4)(1 - u1/3 - u2/6)   (disk integral of the quadratic LD law)
#     catches: wrong LD law, wrong mu, area/visibility mistakes
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,u1,u2,rtol", [(300, 0.29, 0.34, 3e-5), (400, 0.55, 0.15, 6e-5)])
def test_p7_sum_of_weights_limit(N, u1, u2, rtol):
    g = oracle.geometry(star(N=N, u1=u1, u2=u2))
    lim = N * N * (math.pi / 4) * (1 - u1 / 3 - u2 / 6)
    assert abs(g["sum_w"] / lim - 1) < rtol
    assert abs(g["n_visible"] / (N * N * math.pi / 4) - 1) < 2e-4


# ------------------------------------------------------------------------------------------------
# P8: the per-cell operation is numpy.interp(lam*D, lam, S), edge rule included; C oracle == numpy
#     twin on config 1.   catches: off-by-one in the closed-form index, wrong clamp, t vs 1-t
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("v", [-20.0, -2.0, 0.0, 1e-3, 2.0, 20.0, 300.0])
def test_p8_shifted_row_is_numpy_interp(v):
    rng = np.random.default_rng(8)
    P, lam0, k = 3000, 4500.0, 0.01
    S = rng.uniform(0.0, 1.0, P)
    lam = lam0 + k * np.arange(P)
    beta = v / C_KMS
    D = math.sqrt((1 - beta) / (1 + beta))
    got = oracle.shifted_row(S, lam0, k, D)
    # rounding of lam*D (ulp(4500) = 9e-13 A = 9e-11 px) times pixel-to-pixel differences up to 1
    np.testing.assert_allclose(got, np.interp(lam * D, lam, S), rtol=0, atol=3e-10)
    # edges are clamped to the end values
    if v > 0:
        assert got[0] == S[0]
    if v < 0:
        assert got[-1] == S[-1]


def test_p8_c_oracle_equals_numpy_twin_on_config1():
    wl = workloads.make_config1()
    Q, D, na = oracle.run_workload(wl)
    cells = onp.geometry(wl.grid_n, wl.vsini_kms, wl.incl_deg, wl.ld_u1, wl.ld_u2, wl.mu_centres)
    Qn = onp.quiet(cells, wl.quiet, wl.lambda0, wl.dlambda)
    Dn, nan = onp.active(cells, wl.incl_deg, wl.quiet, wl.spot, None, None, None, wl.spot_lb, wl.facula_lb,
                         wl.lambda0, wl.dlambda, wl.regions, wl.phases)
    assert len(cells) == 1976
    # closed-form index vs numpy's bracketing search differ by the ~1e-10 px rounding of lam*D: ~1e-12 relative
    np.testing.assert_allclose(Q, Qn, rtol=1e-11)
    assert list(na) == list(nan)
    assert max(na) > 0
    np.testing.assert_allclose(D, Dn, rtol=0, atol=1e-10 * np.max(np.abs(Dn)))


def test_p8_mu_bins_and_contrast_against_twin():
    """20 mu bins, facula with LB(mu) and a per-pixel contrast, inclination < 90: C oracle == twin."""
    wl = workloads.make_config3(n_pix=600, n_phases=5, grid_n=24)
    wl.incl_deg = 65.0
    wl.vsini_kms = 12.0
    wl.regions = [(-10.0, 150.0, 0.35, 2), (15.0, 200.0, 0.2, 1)]
    Q, D, na = oracle.run_workload(wl)
    cells = onp.geometry(wl.grid_n, wl.vsini_kms, wl.incl_deg, wl.ld_u1, wl.ld_u2, wl.mu_centres)
    assert len({c["bin"] for c in cells}) > 10
    Qn = onp.quiet(cells, wl.quiet, wl.lambda0, wl.dlambda)
    Dn, nan = onp.active(cells, wl.incl_deg, wl.quiet, wl.spot, wl.facula, wl.spot_contrast,
                         wl.facula_contrast, wl.spot_lb, wl.facula_lb, wl.lambda0, wl.dlambda,
                         wl.regions, wl.phases)
    np.testing.assert_allclose(Q, Qn, rtol=1e-11)
    assert list(na) == list(nan) and max(na) > 0
    np.testing.assert_allclose(D, Dn, rtol=0, atol=1e-10 * np.max(np.abs(Dn)))


def test_nearest_bin_rule():
    """'closest mu': nearest centre, tie -> larger mu, clamp outside (reading S9)."""
    st = star(N=300, mu_centres=MU20)
    g = oracle.geometry(st)
    vis = g["visible"] == 1
    mu = g["mu"][vis]
    b = g["bin"][vis]
    expect = np.clip(np.floor(mu / 0.05 + 0.5).astype(int) - 1, 0, 19)
    # closed form for uniform centres, away from exact midpoints
    frac = np.abs((mu / 0.05 + 0.5) % 1.0)
    safe = (frac > 1e-9) & (frac < 1 - 1e-9)
    assert np.array_equal(b[safe], expect[safe])
    assert b.min() == 0 and b.max() == 19
    # non-uniform centres: brute force
    cen = np.array([0.1, 0.15, 0.4, 0.8, 1.0])
    g2 = oracle.geometry(star(N=40, mu_centres=cen))
    v2 = g2["visible"] == 1
    bf = np.argmin(np.abs(g2["mu"][v2][:, None] - cen[None, :]), axis=1)
    assert np.array_equal(g2["bin"][v2], bf)


# ------------------------------------------------------------------------------------------------
# P9: invariants of Eq. 3 / InfoMap
# ------------------------------------------------------------------------------------------------
def _small_active_setup():
    wl = workloads.make_config3(n_pix=800, n_phases=6, grid_n=40)
    wl.vsini_kms = 8.0
    return wl


def _active(wl, regions, phases=None, **kw):
    args = dict(C_spot=wl.spot_contrast, C_facula=wl.facula_contrast, lb_spot=wl.spot_lb, lb_facula=wl.facula_lb)
    args.update(kw)
    return oracle.active(wl, wl.quiet, wl.spot, wl.facula, wl.lambda0, wl.dlambda, regions,
                         wl.phases if phases is None else phases, **args)


def test_p9_linearity_in_spectra():
    wl = _small_active_setup()
    rng = np.random.default_rng(9)
    A = rng.uniform(0, 1, wl.quiet.shape)
    B = rng.uniform(0, 1, wl.quiet.shape)
    qa = oracle.quiet(wl, A, wl.lambda0, wl.dlambda)
    qb = oracle.quiet(wl, B, wl.lambda0, wl.dlambda)
    qab = oracle.quiet(wl, 2.0 * A - 0.5 * B, wl.lambda0, wl.dlambda)
    np.testing.assert_allclose(qab, 2.0 * qa - 0.5 * qb, rtol=0, atol=1e-9)


def test_p9_disjoint_regions_add_and_duplicates_are_idempotent():
    wl = _small_active_setup()
    r1 = (10.0, 150.0, 0.15, 1)
    r2 = (-40.0, 220.0, 0.2, 2)
    ph = np.array([0.45, 0.5, 0.55])
    d1, n1 = _active(wl, [r1], ph)
    d2, n2 = _active(wl, [r2], ph)
    d12, n12 = _active(wl, [r1, r2], ph)
    assert np.all(n1 > 0) and np.all(n2 > 0)
    assert np.array_equal(n12, n1 + n2)
    np.testing.assert_allclose(d12, d1 + d2, rtol=0, atol=1e-10 * np.abs(d12).max())
    dd, nd = _active(wl, [r1, r1, r2, r2], ph)
    assert np.array_equal(nd, n12)
    np.testing.assert_array_equal(dd, d12)


def test_p9_later_region_overrides():
    wl = _small_active_setup()
    fac = (20.0, 180.0, 0.3, 2)
    spot = (20.0, 180.0, 0.1, 1)
    ph = np.array([0.5])
    d_fs, n_fs = _active(wl, [fac, spot], ph)   # spot embedded in facula
    d_sf, n_sf = _active(wl, [spot, fac], ph)   # facula listed last covers the spot entirely
    d_f, n_f = _active(wl, [fac], ph)
    assert n_fs[0] == n_f[0] == n_sf[0]
    np.testing.assert_array_equal(d_sf, d_f)
    assert np.abs(d_fs - d_f).max() > 1e-3 * np.abs(d_f).max()
    # type maps: spot cells are a strict subset carrying type 1
    tm, _ = oracle.info_map(wl, [fac, spot], 0.5)
    tms, ns = oracle.info_map(wl, [spot], 0.5)
    assert ns > 0 and np.all(tm[tms == 1] == 1) and np.sum(tm == 2) == n_f[0] - ns


def test_p9_identical_spectrum_gives_zero_delta():
    wl = _small_active_setup()
    d, n = oracle.active(wl, wl.quiet, wl.quiet, wl.quiet, wl.lambda0, wl.dlambda,
                         [(0.0, 180.0, 0.2, 1), (30.0, 100.0, 0.2, 2)], np.array([0.4, 0.5]))
    assert np.all(n > 0)
    assert np.abs(d).max() == 0.0


def test_p9_far_side_region_gives_exact_zero_and_lon180_crosses_centre_at_half_phase():
    wl = _small_active_setup()
    reg = [(0.0, 180.0, 0.1, 1)]
    d, n = _active(wl, reg, np.array([0.0, 0.5]))
    assert n[0] == 0 and np.all(d[0] == 0.0)
    assert n[1] > 0
    tm, _ = oracle.info_map(wl, reg, 0.5)
    g = oracle.geometry(wl)
    act = np.flatnonzero(tm)
    # the covered cells are centred on the disk centre ("crosses the center of the disk (phase=0.5)")
    assert abs(g["x"][act].mean()) < 1e-12 and abs(g["y"][act].mean()) < 1e-12
    # and a region moves toward +x (the receding limb) with increasing phase
    tm2, _ = oracle.info_map(wl, reg, 0.55)
    assert g["x"][np.flatnonzero(tm2)].mean() > 0.1


def test_p9_inclination_tilts_north_pole_toward_observer():
    """Reading S13: for i < 90 deg a region at positive latitude on the central meridian moves DOWN... no:
    y_r = sin(lat) sin(i) - cos(lat) cos(i); at lat = 90 - i the region sits at the disk centre."""
    st = star(N=60, incl=60.0)
    tm, n = oracle.info_map(st, [(30.0, 0.0, 0.1, 1)], 0.0)
    g = oracle.geometry(st)
    act = np.flatnonzero(tm)
    assert n > 0 and abs(g["y"][act].mean()) < 1e-12 and abs(g["x"][act].mean()) < 1e-12
    # the pole itself is visible, at y = cos(i)... i.e. (0, sin(90)sin(60)) = +0.866 above centre
    tm, n = oracle.info_map(st, [(90.0, 0.0, 0.1, 1)], 0.3)
    act = np.flatnonzero(tm)
    assert n > 0 and abs(g["y"][act].mean() - math.sin(math.radians(60.0))) < 0.02


def test_p9_redshifted_quiet_as_spot_gives_one_signed_rv():
    """The paper's own sanity experiment: injecting the quiet spectrum red-shifted by 300 m/s as
    the active spectrum (contrast 1) gives a convective-blueshift-inhibition RV that never goes negative."""
    P, lam0, k = 3000, 5000.0, 0.01
    lam = lam0 + k * np.arange(P)
    centres = np.array([5008.0, 5015.0, 5022.0])
    z = 0.300 / C_KMS
    Sq = np.tile(gaussian_spectrum(P, lam0, k, centres, [0.5, 0.7, 0.3], [0.05, 0.04, 0.06]), (20, 1))
    Sa = np.tile(gaussian_spectrum(P, lam0, k, centres * (1 + z), [0.5, 0.7, 0.3], [0.05, 0.04, 0.06]), (20, 1))
    st = star(N=80, mu_centres=MU20)
    ph = np.linspace(0.3, 0.7, 9)
    D, n = oracle.active(st, Sq, Sa, None, lam0, k, [(0.0, 180.0, 0.2, 1)], ph)
    Q = oracle.quiet(st, Sq, lam0, k)
    sw = oracle.geometry(st)["sum_w"]
    assert np.all(n > 0)
    for c in centres:
        win = np.abs(lam - c) < 0.3
        rv0 = np.sum((lam - c)[win] * (1 - Q[win] / sw)) / np.sum(1 - Q[win] / sw)
        for p in range(len(ph)):
            F = Q + D[p]
            rv = np.sum((lam - c)[win] * (1 - F[win] / sw)) / np.sum(1 - F[win] / sw)
            assert rv - rv0 > 0.0


# ------------------------------------------------------------------------------------------------
# P10: the direct index u = (lam D - lam0)/k and the shift form m + (D-1)(lam0/k + m) agree
#      (guards the oracle's own index arithmetic against cancellation)
# ------------------------------------------------------------------------------------------------
def test_p10_direct_and_shift_form_index_agree():
    rng = np.random.default_rng(10)
    P, lam0, k = 310_000, 3800.0, 0.01
    S = rng.uniform(0.5, 1.0, P)
    m = np.arange(2000, P - 2000, 997)
    for v in (2.0, -2.0, 20.0):
        beta = v / C_KMS
        D = math.sqrt((1 - beta) / (1 + beta))
        dm1 = -2 * beta / ((1 + beta) + math.sqrt(1 - beta * beta))  # D - 1 without cancellation
        assert abs((D - 1) - dm1) < 1e-15
        u = m + dm1 * (lam0 / k + m)
        n = np.floor(u).astype(np.int64)
        t = u - n
        alt = S[n] + t * (S[n + 1] - S[n])
        got = np.array([oracle.shifted_row(S, lam0, k, D, int(mm), int(mm) + 1)[0] for mm in m])
        assert np.max(np.abs(got - alt)) < 5e-10


def test_oracle_is_thread_count_invariant():
    wl = workloads.make_config2(n_pix=5000, n_phases=3, grid_n=60)
    n0 = oracle.num_threads()
    try:
        oracle.set_threads(1)
        q1 = oracle.quiet(wl, wl.quiet, wl.lambda0, wl.dlambda)
        oracle.set_threads(max(2, n0))
        q2 = oracle.quiet(wl, wl.quiet, wl.lambda0, wl.dlambda)
    finally:
        oracle.set_threads(n0)
    np.testing.assert_array_equal(q1, q2)


def test_sub_range_equals_full_range():
    wl = workloads.make_config2(n_pix=6000, n_phases=4, grid_n=50)
    wl.phases = np.array([0.4, 0.5, 0.6, 0.0])
    Q, D, na = oracle.run_workload(wl)
    Qs, Ds, nas = oracle.run_workload(wl, 2500, 4700)
    np.testing.assert_array_equal(Q[2500:4700], Qs)
    np.testing.assert_array_equal(D[:, 2500:4700], Ds)
    np.testing.assert_array_equal(na, nas)
