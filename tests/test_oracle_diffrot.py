"""Pins of the oracle's differential rotation (Fig. 1; reading R-DR).

omega = omega_0 + omega_1 sin^2(latitude); the oracle's parameter is diff_rot = omega_1 / omega_0 (-0.18 for the
Sun: -2.587 / 14.371).  The pins are closed forms of the velocity field and consistency with the region geometry,
not a second copy of the oracle's line."""
from __future__ import annotations

import math
from types import SimpleNamespace

import numpy as np
import pytest

import oracle
from oracle import soap_oracle_np as onp
import workloads

C_KMS = 299792.458


def star(N=60, vsini=2.0, incl=90.0, dr=0.0, u1=0.0, u2=0.0):
    return SimpleNamespace(grid_n=N, vsini_kms=vsini, incl_deg=incl, ld_u1=u1, ld_u2=u2, mu_centres=np.array([1.0]),
                           doppler_mode=0, diff_rot=dr)


def test_zero_rate_is_solid_body_bit_for_bit():
    a, b = oracle.geometry(star(dr=0.0, incl=63.0)), oracle.geometry(star(incl=63.0))
    np.testing.assert_array_equal(a["vel"], b["vel"])
    np.testing.assert_array_equal(a["D"], b["D"])


def test_equator_on_velocity_field_closed_form():
    """i = 90: latitude = asin(y), so v = x vsini (1 + dr y^2): iso-velocity lines are not vertical (Fig. 1)."""
    g = oracle.geometry(star(N=40, vsini=3.0, dr=-0.18))
    vis = g["visible"] == 1
    np.testing.assert_allclose(g["vel"][vis], (g["x"] * 3.0 * (1.0 - 0.18 * g["y"] ** 2))[vis], rtol=1e-14, atol=1e-16)
    col = g["vel"].reshape(40, 40)[33]          # one column, x > 0: fastest on the equator, slower toward the poles
    v = col[g["visible"].reshape(40, 40)[33] == 1]
    assert v.argmax() in (len(v) // 2 - 1, len(v) // 2) and v[0] < v.max() and v[-1] < v.max()


@pytest.mark.parametrize("dr", [-0.18, 0.3])
def test_velocity_second_moment_converges_to_disk_integral(dr):
    """<v^2> / vsini^2 over the unit disk = <x^2 (1 + dr y^2)^2> = 1/4 + dr/12 + dr^2/64 (i = 90, no weights)."""
    g = oracle.geometry(star(N=400, vsini=2.0, dr=dr))
    vis = g["visible"] == 1
    m2 = float(np.mean(g["vel"][vis] ** 2)) / 4.0
    assert abs(m2 / (0.25 + dr / 12.0 + dr * dr / 64.0) - 1.0) < 2e-4


def test_pole_on_star_does_not_shift_and_inclined_latitudes_match_the_region_frame():
    g = oracle.geometry(star(N=30, vsini=5.0, incl=0.0, dr=-0.2))
    assert np.max(np.abs(g["vel"])) < 1e-15 * 5.0 + 1e-15
    # the surface point a region centre (lat, lon) projects to (reading S13, pinned by P9) rotates at
    # omega_0 (1 + dr sin^2 lat): compare the nearest cell of a fine grid
    N, incl, dr = 600, 55.0, -0.25
    g = oracle.geometry(star(N=N, vsini=4.0, incl=incl, dr=dr))
    x, y, v = g["x"].reshape(N, N), g["y"].reshape(N, N), g["vel"].reshape(N, N)
    for lat, lon in [(40.0, 25.0), (-30.0, -50.0), (70.0, 10.0), (0.0, 60.0)]:
        xr, yr, zr = onp.region_centre(lat, lon, incl, 0.0)
        assert zr > 0.1
        j, i = int(round((xr + 1) * N / 2 - 0.5)), int(round((yr + 1) * N / 2 - 0.5))
        ratio = v[j, i] / (x[j, i] * 4.0 * math.sin(math.radians(incl)))
        assert abs(ratio - (1.0 + dr * math.sin(math.radians(lat)) ** 2)) < 3e-3   # cell centre within 1/N of the point


def test_linear_spectrum_closed_form_with_per_cell_doppler_factors():
    """S = a + b lambda  =>  Q[m] = a sum w + b lambda_m sum_c w_c D_c in the interior, D_c from the closed-form field."""
    st = star(N=50, vsini=12.0, dr=-0.18, u1=0.3, u2=0.2)
    P, lam0, k = 1500, 5000.0, 0.01
    lam = lam0 + k * np.arange(P)
    a, b = 0.4, 1e-4
    Q = oracle.quiet(st, (a + b * lam)[None, :], lam0, k)
    g = oracle.geometry(st)
    vis = g["visible"] == 1
    beta = (g["x"] * 12.0 * (1.0 - 0.18 * g["y"] ** 2))[vis] / C_KMS
    D = np.sqrt((1 - beta) / (1 + beta))
    w = g["w"][vis]
    expect = a * w.sum() + b * lam * float(np.sum(w * D))
    np.testing.assert_allclose(Q[20:-20], expect[20:-20], rtol=1e-12)


def test_differential_rotation_narrows_or_widens_a_line_as_the_second_moment_says():
    """The rotational broadening adds (lambda / c)^2 <v^2>_w to a line's variance: slower high latitudes (dr < 0)
    give a narrower line than solid-body rotation, faster ones (dr > 0) a broader line."""
    P, lam0, k, lc = 4000, 5000.0, 0.01, 5020.0
    lam = lam0 + k * np.arange(P)
    S = (1.0 - 0.5 * np.exp(-(lam - lc) ** 2 / (2 * 0.05 ** 2)))[None, :]
    var = {}
    for dr in (-0.3, 0.0, 0.3):
        st = star(N=120, vsini=20.0, dr=dr)
        Q = oracle.quiet(st, S, lam0, k)
        g = oracle.geometry(st)
        dep = 1.0 - Q / g["sum_w"]
        mean = float((lam * dep).sum() / dep.sum())
        var[dr] = float(((lam - mean) ** 2 * dep).sum() / dep.sum())
        vis = g["visible"] == 1
        expect = 0.05 ** 2 + (lc / C_KMS) ** 2 * float(np.mean(g["vel"][vis] ** 2)) + k * k / 6.0  # + lerp smoothing (pin P4)
        assert abs(var[dr] / expect - 1.0) < 2e-3
    assert var[-0.3] < var[0.0] < var[0.3]


def test_c_oracle_equals_numpy_twin_with_differential_rotation():
    wl = workloads.make_config3(n_pix=500, n_phases=4, grid_n=22)
    wl.incl_deg, wl.vsini_kms, wl.diff_rot = 60.0, 15.0, -0.18
    wl.regions = [(-10.0, 150.0, 0.35, 2), (15.0, 200.0, 0.2, 1)]
    Q, D, na = oracle.run_workload(wl)
    cells = onp.geometry(wl.grid_n, wl.vsini_kms, wl.incl_deg, wl.ld_u1, wl.ld_u2, wl.mu_centres, diff_rot=wl.diff_rot)
    Qn = onp.quiet(cells, wl.quiet, wl.lambda0, wl.dlambda)
    Dn, nan = onp.active(cells, wl.incl_deg, wl.quiet, wl.spot, wl.facula, wl.spot_contrast, wl.facula_contrast,
                         wl.spot_lb, wl.facula_lb, wl.lambda0, wl.dlambda, wl.regions, wl.phases)
    np.testing.assert_allclose(Q, Qn, rtol=1e-11)
    assert list(na) == list(nan) and max(na) > 0
    np.testing.assert_allclose(D, Dn, rtol=0, atol=1e-10 * np.max(np.abs(Dn)))
    # and it is not the solid-body answer
    wl.diff_rot = 0.0
    assert np.max(np.abs(oracle.run_workload(wl)[0] - Q)) > 1e-3
