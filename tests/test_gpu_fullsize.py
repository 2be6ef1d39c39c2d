"""BASELINE.json's full-size configurations compared with the fp64 oracle on EVERY pixel and EVERY line.  -m gpu.

north_star's target sentence is about the whole C3 time series: quiet <= 1e-5 of the integrated continuum, deltas
<= 1e-4 of max|delta|, first-moment RV of each of the 25 000 generated lines in each of the 26 spectra within 1 cm/s.
The sampled-window tests of test_gpu_parity.py stay as quick checks; these run the oracle over all pixels (C3: ~3.5e10
fp64 lerps, tens of seconds on the box's host cores), once per workload (module-scoped fixtures), and compare every
form of the CUDA path with it.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import workloads
from helpers import DELTA_TOL, QUIET_TOL, RV_TOL_CMS, check_delta, check_quiet, line_rvs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

FORM_BINNED, FORM_FIR, FORM_COMPOSITE = 1, 3, 4


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


def _oracle_all(wl):
    Qo, Do, nao = oracle.run_workload(wl)
    sw = oracle.geometry(wl)["sum_w"]
    # the oracle's own line RVs, for Q and for Q + delta_p of every phase: [1 + n_phases, n_lines]
    F = np.concatenate([Qo[None, :], Qo[None, :] + Do], axis=0)
    rv = line_rvs(F, sw, wl.lambda0, wl.dlambda, wl.line_centres, wl.line_sigmas, 0, 64)
    return dict(Q=Qo, D=Do, n_active=nao, sum_w=sw, rv=rv)


@pytest.fixture(scope="module")
def c3():
    wl = workloads.make_config3()
    return wl, _oracle_all(wl)


def _run(soap, wl, form=None):
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    if form is not None:
        soap.soap_set_option(star, soap.binding.SOAP_OPT_FORM, form)
    soap.soap_disk_geometry(star, wl)
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    s = None if wl.spot is None else soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    f = None if wl.facula is None else soap.to_device_spectra(wl.facula, wl.lambda0, wl.dlambda, dev, wl.facula_contrast, wl.facula_lb)
    Q = torch.full((wl.n_pix,), float("nan"), dtype=torch.float32, device=dev)
    D = torch.full((len(wl.phases), wl.n_pix), float("nan"), dtype=torch.float32, device=dev)
    soap.soap_integrate_quiet(star, q, Q)
    na = soap.soap_active_timeseries(star, q, s, f, wl.regions, wl.phases, D, want_n_active=True)
    torch.cuda.synchronize()
    stats = soap.soap_get_stats(star)
    soap.soap_destroy(star)
    return Q.cpu().numpy(), D.cpu().numpy(), na, stats


def _assert_every_pixel_and_line(wl, ref, Q, D, na):
    assert not np.isnan(Q).any() and not np.isnan(D).any(), "every pixel of every row must be written"
    eq = check_quiet(Q, ref["Q"], ref["sum_w"])
    assert eq <= QUIET_TOL, f"quiet: {eq:.3e} of continuum"
    ed = check_delta(D, ref["D"])
    assert ed <= DELTA_TOL, f"delta: {ed:.3e} of max|delta|"
    assert np.array_equal(na, ref["n_active"])
    for p in np.nonzero(ref["n_active"] == 0)[0]:
        assert np.all(D[p] == 0.0), "empty phase must be exact zeros"
    Q64 = Q.astype(np.float64)
    F = np.concatenate([Q64[None, :], Q64[None, :] + D.astype(np.float64)], axis=0)
    rv = line_rvs(F, ref["sum_w"], wl.lambda0, wl.dlambda, wl.line_centres, wl.line_sigmas, 0, 64)
    d = np.abs(rv - ref["rv"])
    n_checked = int(np.sum(~np.isnan(d)))
    assert n_checked >= 0.99 * d.size, "nearly every line lies inside the grid"
    worst = float(np.nanmax(d))
    assert worst <= RV_TOL_CMS, f"line RV differs by {worst:.3f} cm/s over {n_checked} (spectrum, line) pairs"
    return eq, ed, worst


def test_config3_every_pixel_every_line_binned(soap, c3):
    wl, ref = c3
    Q, D, na, stats = _run(soap, wl, FORM_BINNED)
    assert stats["form"] == FORM_BINNED
    assert int(na.sum()) == 20650 and na.max() == 1920
    _assert_every_pixel_and_line(wl, ref, Q, D, na)


def test_config3_every_pixel_every_line_auto(soap, c3):
    """Whatever form SOAP_FORM_AUTO picks - the configuration bench.py times."""
    wl, ref = c3
    Q, D, na, _ = _run(soap, wl, None)
    _assert_every_pixel_and_line(wl, ref, Q, D, na)


def test_config3_every_pixel_every_line_fir(soap, c3):
    wl, ref = c3
    Q, D, na, stats = _run(soap, wl, FORM_FIR)
    assert stats["form"] == FORM_FIR
    _assert_every_pixel_and_line(wl, ref, Q, D, na)


def test_config3_every_pixel_every_line_composite(soap, c3):
    wl, ref = c3
    Q, D, na, stats = _run(soap, wl, FORM_COMPOSITE)
    assert stats["form"] == FORM_COMPOSITE
    _assert_every_pixel_and_line(wl, ref, Q, D, na)


def test_config3_differential_rotation_every_pixel_every_line(soap):
    wl = workloads.make_config3()
    wl.diff_rot = -0.18
    ref = _oracle_all(wl)
    Q, D, na, _ = _run(soap, wl, None)
    _assert_every_pixel_and_line(wl, ref, Q, D, na)


def test_config4_every_pixel_every_line(soap):
    wl = workloads.make_config4()
    ref = _oracle_all(wl)
    Q, D, na, _ = _run(soap, wl, None)
    _assert_every_pixel_and_line(wl, ref, Q, D, na)


def test_config3_nested_spot_in_facula_every_pixel_every_line(soap):
    """The spot-inside-a-facula variant of C3 (list order decides, the spot listed after the facula overrides it)."""
    wl = workloads.make_config3(nested=True)
    ref = _oracle_all(wl)
    Q, D, na, _ = _run(soap, wl, None)
    assert int(na.sum()) == 14694 and na.max() == 1825
    _assert_every_pixel_and_line(wl, ref, Q, D, na)


def test_config3_three_effects_in_one_pass_every_pixel(soap, c3):
    """Total, flux-only and CB-only delta spectra (Eq. 1-3) from the one-pass launch on C3 as configured (the facula has a
    limb-brightening law, so its entries are walked with both weights): every pixel of every phase of the three outputs against
    the oracle's three effects, each held to 1e-4 of its own max|delta| and never looser than 1e-4 of the total's."""
    from test_gpu_parity import _run_effects
    wl, ref = c3
    outs, na = _run_effects(soap, wl)
    assert np.array_equal(na, ref["n_active"])
    scale = float(np.max(np.abs(ref["D"])))
    for effect, D in enumerate(outs):
        assert not np.isnan(D).any()
        if effect == 0:
            Do = ref["D"]
        else:
            Do, nao = oracle.active(wl, wl.quiet, wl.spot, wl.facula, wl.lambda0, wl.dlambda, wl.regions, wl.phases,
                                    wl.spot_contrast, wl.facula_contrast, wl.spot_lb, wl.facula_lb, 0, None, effect)
            assert np.array_equal(nao, ref["n_active"])
        own = float(np.max(np.abs(Do)))
        assert own > 0
        err = float(np.max(np.abs(D.astype(np.float64) - Do)))
        assert err <= DELTA_TOL * min(own, scale), f"effect {effect}: {err / min(own, scale):.3e} of max|delta|"
        for p_ in np.nonzero(ref["n_active"] == 0)[0]:
            assert np.all(D[p_] == 0.0)


def test_config5_batch_all_stars_16k_pixel_windows(soap):
    """64 stars through the batch entry points; the slowest and fastest rotator, the most pole-on and most equator-on star,
    the stars with the most and the fewest regions and the first and last star are compared with the oracle on three
    16 384-pixel windows each: both ends of the spectrum (clamped halo) and a stretch across tile boundaries; every other
    star on one window whose position moves along the spectrum with the star's index."""
    dev = torch.device("cuda:0")
    n_stars, n_pix, n_ph = 64, 200_000, 50
    shared = workloads.make_config5_star(0, n_pix=n_pix, n_phases=n_ph)
    wls = [shared] + [workloads.make_config5_star(k, n_pix=n_pix, n_phases=n_ph, shared=shared) for k in range(1, n_stars)]
    q = soap.to_device_spectra(shared.quiet, shared.lambda0, shared.dlambda, dev)
    s = soap.to_device_spectra(shared.spot, shared.lambda0, shared.dlambda, dev, shared.spot_contrast, shared.spot_lb)
    f = soap.to_device_spectra(shared.facula, shared.lambda0, shared.dlambda, dev, shared.facula_contrast, shared.facula_lb)
    stars = [soap.soap_create(0) for _ in range(n_stars)]
    for st, wl in zip(stars, wls):
        soap.soap_disk_geometry(st, wl, want_info=False)
    Q = torch.full((n_stars, n_pix), float("nan"), dtype=torch.float32, device=dev)
    D = torch.full((n_stars, n_ph, n_pix), float("nan"), dtype=torch.float32, device=dev)
    soap.soap_batch_integrate_quiet(stars, [q] * n_stars, [Q[k] for k in range(n_stars)])
    soap.soap_batch_active_timeseries(stars, [q] * n_stars, [s] * n_stars, [f] * n_stars, [w.regions for w in wls],
                                      [w.phases for w in wls], [D[k] for k in range(n_stars)])
    torch.cuda.synchronize()
    assert not torch.isnan(Q).any() and not torch.isnan(D).any()
    vs = [w.vsini_kms for w in wls]
    inc = [w.incl_deg for w in wls]
    nr = [len(w.regions) for w in wls]
    picks = sorted({0, n_stars - 1, int(np.argmax(vs)), int(np.argmin(vs)), int(np.argmin(inc)), int(np.argmax(inc)),
                    int(np.argmax(nr)), int(np.argmin(nr))})
    if len(picks) < 8:
        picks = sorted(set(picks) | set(range(1, 64, 9)))[:max(8, len(picks))]
    W = 16384
    for k in range(n_stars):
        wl = wls[k]
        Qk, Dk = Q[k].cpu().numpy(), D[k].cpu().numpy()
        sw = oracle.geometry(wl)["sum_w"]
        windows = (0, 96_000, n_pix - W) if k in picks else ((k * 2897) % ((n_pix - W) // 64) * 64,)
        for lo in windows:
            hi = lo + W
            Qo, Do, _ = oracle.run_workload(wl, lo, hi)
            assert check_quiet(Qk[lo:hi], Qo, sw) <= QUIET_TOL, f"star {k} window {lo}"
            if np.abs(Do).max() > 0:
                assert check_delta(Dk[:, lo:hi], Do) <= DELTA_TOL, f"star {k} window {lo}"
            else:
                assert np.all(Dk[:, lo:hi] == 0.0)
            Fg = np.concatenate([Qk[None, lo:hi].astype(np.float64), Qk[None, lo:hi].astype(np.float64) + Dk[:, lo:hi]], axis=0)
            Fo = np.concatenate([Qo[None, :], Qo[None, :] + Do], axis=0)
            a = line_rvs(Fg, sw, wl.lambda0, wl.dlambda, wl.line_centres, wl.line_sigmas, lo, 64)
            b = line_rvs(Fo, sw, wl.lambda0, wl.dlambda, wl.line_centres, wl.line_sigmas, lo, 64)
            d = np.abs(a - b)
            assert np.sum(~np.isnan(d)) > 0 and float(np.nanmax(d)) <= RV_TOL_CMS, f"star {k} window {lo}: {np.nanmax(d):.3f} cm/s"
    for st in stars:
        soap.soap_destroy(st)
