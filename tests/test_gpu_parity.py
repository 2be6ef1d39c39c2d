"""Parity of the CUDA path (through the C ABI) against the fp64 CPU oracle.  Needs a B200: -m gpu.

Tolerances are BASELINE.json north_star's: quiet <= 1e-5 of the integrated continuum, deltas <= 1e-4 of
max|delta|, per-line first-moment RV within 1 cm/s; integer outputs (bins, visible cells, active-cell
counts) bit-exact.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import workloads
from helpers import DELTA_TOL, QUIET_TOL, RV_TOL_CMS, check_delta, check_quiet, max_rv_diff

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


def run_gpu(soap, wl, form=None, splits=None, want_n_active=True):
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    if form is not None:
        soap.soap_set_option(star, soap.binding.SOAP_OPT_FORM, form)
    if splits is not None:
        soap.soap_set_option(star, soap.binding.SOAP_OPT_QUIET_SPLITS, splits)
    info = soap.soap_disk_geometry(star, wl)
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    s = None if wl.spot is None else soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    f = None if wl.facula is None else soap.to_device_spectra(wl.facula, wl.lambda0, wl.dlambda, dev, wl.facula_contrast, wl.facula_lb)
    tdt = torch.float32 if wl.dtype == np.float32 else torch.float64
    Q = torch.full((wl.n_pix,), float("nan"), dtype=tdt, device=dev)
    soap.soap_integrate_quiet(star, q, Q)
    n_ph = len(wl.phases)
    D = torch.full((n_ph, wl.n_pix), float("nan"), dtype=tdt, device=dev)
    na = soap.soap_active_timeseries(star, q, s, f, wl.regions, wl.phases, D, want_n_active=want_n_active)
    torch.cuda.synchronize()
    stats = soap.soap_get_stats(star)
    geo = soap.soap_export_geometry(star, wl.grid_n)
    soap.soap_destroy(star)
    return dict(Q=Q.cpu().numpy(), D=D.cpu().numpy(), n_active=na, info=info, stats=stats, geo=geo)


def assert_parity(wl, g, m_lo=0, m_hi=None, check_rv=True):
    Qo, Do, nao = oracle.run_workload(wl, m_lo, m_hi)
    sw = oracle.geometry(wl)["sum_w"]
    sl = slice(m_lo, m_hi)
    eq = check_quiet(g["Q"][sl], Qo, sw)
    assert eq <= QUIET_TOL, f"quiet: {eq:.3e} of continuum"
    ed = check_delta(g["D"][:, sl], Do)
    assert ed <= DELTA_TOL, f"delta: {ed:.3e} of max|delta|"
    assert np.array_equal(g["n_active"], nao)
    for p in range(len(wl.phases)):
        if nao[p] == 0:
            assert np.all(g["D"][p] == 0.0), "empty phase must be exact zeros"
    if check_rv and len(wl.line_centres):
        rvq, n_lines = max_rv_diff(g["Q"][sl].astype(np.float64), Qo, sw, wl, m_lo)
        assert rvq <= RV_TOL_CMS, f"quiet line RV differs by {rvq:.3f} cm/s over {n_lines} lines"
        F_gpu = g["Q"][sl].astype(np.float64)[None, :] + g["D"][:, sl].astype(np.float64)
        rvd, _ = max_rv_diff(F_gpu, Qo[None, :] + Do, sw, wl, m_lo)
        assert rvd <= RV_TOL_CMS, f"Q+delta line RV differs by {rvd:.3f} cm/s"
    return eq, ed


def test_geometry_matches_oracle_exactly(soap):
    wl = workloads.make_config2(n_pix=2000, n_phases=2)
    g = run_gpu(soap, wl)
    og = oracle.geometry(wl)
    assert g["info"]["n_visible"] == og["n_visible"] == 70688
    assert np.array_equal(g["geo"]["bin"], og["bin"])
    np.testing.assert_array_equal(g["geo"]["mu"], og["mu"])
    np.testing.assert_array_equal(g["geo"]["w"], og["w"])
    np.testing.assert_array_equal(g["geo"]["vel"], og["vel"])
    assert abs(g["info"]["sum_weights"] / og["sum_w"] - 1) < 1e-13
    assert g["info"]["n_entries"] == len({(c // 300, b) for c, b in enumerate(og["bin"]) if b >= 0}) == 4554


def test_config1_fp64(soap):
    wl = workloads.make_config1()
    g = run_gpu(soap, wl)
    Qo, Do, nao = oracle.run_workload(wl)
    sw = oracle.geometry(wl)["sum_w"]
    # fp64 end to end: only the ~5e-12 px difference between the oracle's direct source coordinate and the
    # kernel's shift form (pin P10) is left
    assert check_quiet(g["Q"], Qo, sw) <= 1e-10
    assert check_delta(g["D"], Do) <= 1e-9
    assert np.array_equal(g["n_active"], nao) and nao.max() > 0
    assert_parity(wl, g)


def test_config1_paper_phases(soap):
    """BASELINE.json's literal '4 phases evenly over one rotation' {0, 1/4, 1/2, 3/4}: only 1/2 is active."""
    wl = workloads.make_config1(phases=np.array([0.0, 0.25, 0.5, 0.75]))
    g = run_gpu(soap, wl)
    assert list(g["n_active"]) == [0, 0, 16, 0]
    assert_parity(wl, g)


def test_config2_full(soap):
    wl = workloads.make_config2()
    g = run_gpu(soap, wl)
    assert g["n_active"].max() == 668 and int(g["n_active"].sum()) == 21178
    assert_parity(wl, g)


@pytest.mark.parametrize("form", [1, 2, 3])
def test_forms_agree_with_oracle(soap, form):
    """Pre-binned (column, mu-bin) entries, the literal one-entry-per-cell form, and the run-collapsed (FIR) form."""
    wl = workloads.make_config2(n_pix=3000, n_phases=8, grid_n=120)
    wl.phases = np.linspace(0.3, 0.7, 8)
    g = run_gpu(soap, wl, form=form)
    assert g["stats"]["form"] == form
    assert_parity(wl, g)


@pytest.mark.parametrize("n_pix", [2, 3, 5, 127, 1023, 1024, 1025, 4099])
def test_ragged_sizes(soap, n_pix):
    wl = workloads.make_config2(n_pix=max(n_pix, 400), n_phases=3, grid_n=40)
    # cut the arrays down to n_pix (keeps line structure near the start)
    wl.n_pix = n_pix
    wl.quiet = np.ascontiguousarray(wl.quiet[:, :n_pix])
    wl.spot = np.ascontiguousarray(wl.spot[:, :n_pix])
    wl.spot_contrast = np.ascontiguousarray(wl.spot_contrast[:n_pix])
    wl.phases = np.array([0.45, 0.5, 0.0])
    wl.vsini_kms = 25.0
    g = run_gpu(soap, wl)
    assert_parity(wl, g, check_rv=False)


def test_fast_rotator_large_halo_and_inclination(soap):
    wl = workloads.make_config5_star(3, n_pix=6000, n_phases=6, grid_n=90)
    wl.vsini_kms = 20.0
    wl.incl_deg = 35.0
    wl.regions = [(20.0, 170.0, 0.25, 2), (25.0, 175.0, 0.1, 1), (-30.0, 30.0, 0.15, 1)]
    wl.phases = np.linspace(0.0, 1.0, 6, endpoint=False)
    g = run_gpu(soap, wl)
    assert_parity(wl, g)


def test_first_order_doppler_mode(soap):
    wl = workloads.make_config2(n_pix=3000, n_phases=2, grid_n=60)
    wl.vsini_kms = 20.0
    wl.doppler_mode = 1
    wl.phases = np.array([0.5, 0.55])
    g = run_gpu(soap, wl)
    assert_parity(wl, g)


def test_nonuniform_mu_centres_and_facula_contrast(soap):
    wl = workloads.make_config3(n_pix=2500, n_phases=4, grid_n=80, nested=True)
    wl.mu_centres = np.array([0.1, 0.3, 0.35, 0.6, 0.9, 1.0])
    wl.quiet, wl.spot, wl.facula = (np.ascontiguousarray(a[:6]) for a in (wl.quiet, wl.spot, wl.facula))
    wl.facula_contrast = (1.0 + 0.05 * np.sin(np.arange(wl.n_pix) / 50.0)).astype(np.float32)
    wl.phases = np.array([0.4, 0.5, 0.6, 0.9])
    g = run_gpu(soap, wl)
    assert_parity(wl, g)


def test_splits_do_not_change_parity_and_runs_are_deterministic(soap):
    wl = workloads.make_config2(n_pix=5000, n_phases=4, grid_n=100)
    wl.phases = np.array([0.4, 0.5, 0.6, 0.0])
    a = run_gpu(soap, wl, splits=1)
    b = run_gpu(soap, wl, splits=7)
    c = run_gpu(soap, wl, splits=7)
    assert_parity(wl, a)
    assert_parity(wl, b)
    assert np.array_equal(b["Q"], c["Q"]) and np.array_equal(b["D"], c["D"])


@pytest.mark.parametrize("which", ["facula_only", "spot_only", "neither", "both"])
def test_contrast_array_on_either_kind_or_none(soap, which):
    """A per-pixel contrast on the spot rows only, the facula rows only, both or neither (NULL == 1, soap_b200.h):
    the kinds of one phase are summed in the order spot, facula, quiet and each sum takes only its own contrast."""
    wl = workloads.make_config3(n_pix=5000, n_phases=4, grid_n=90)
    wl.regions = [(-25.0, 170.0, 0.25, 2), (20.0, 185.0, 0.15, 1)]   # both kinds visible together, not nested
    wl.phases = np.array([0.45, 0.5, 0.55, 0.0])
    ramp = np.arange(wl.n_pix, dtype=np.float64) / wl.n_pix
    wl.spot_contrast = (0.3 + 0.2 * ramp).astype(np.float32) if which in ("spot_only", "both") else None
    wl.facula_contrast = (1.2 - 0.15 * ramp).astype(np.float32) if which in ("facula_only", "both") else None
    g = run_gpu(soap, wl)
    assert g["n_active"][:3].min() > 0
    assert_parity(wl, g)


def test_overlap_override_and_duplicates(soap):
    wl = workloads.make_config3(n_pix=2000, n_phases=3, grid_n=100, nested=True)
    wl.phases = np.array([0.45, 0.5, 0.55])
    g1 = run_gpu(soap, wl)
    assert_parity(wl, g1)
    wl2 = workloads.make_config3(n_pix=2000, n_phases=3, grid_n=100, nested=True)
    wl2.phases = wl.phases
    wl2.regions = [wl.regions[0], wl.regions[0], wl.regions[1], wl.regions[1]]
    g2 = run_gpu(soap, wl2)
    assert np.array_equal(g1["D"], g2["D"]) and np.array_equal(g1["n_active"], g2["n_active"])


def test_no_regions_and_zero_rotation(soap):
    wl = workloads.make_config2(n_pix=1500, n_phases=2, grid_n=50)
    wl.regions = []
    wl.vsini_kms = 0.0
    g = run_gpu(soap, wl)
    assert np.all(g["D"] == 0.0) and np.all(g["n_active"] == 0)
    assert_parity(wl, g)


# ---- BASELINE.json full sizes, in the launch configuration bench.py times: sampled pixel ranges ----
def _sample_ranges(n_pix, width=768, n=6):
    rng = np.random.default_rng(123)
    starts = [0, n_pix - width] + [int(v) for v in rng.integers(2048, n_pix - width - 2048, n)]
    # make two of them straddle a tile boundary (f32::kTile = 2048 px; the library reports it as stats.tile_px)
    starts[2] = 2048 * (starts[2] // 2048) - width // 2
    starts[3] = 2048 * (starts[3] // 2048) - 3
    return [(s, s + width) for s in starts]


def test_config3_full_size_sampled(soap):
    wl = workloads.make_config3()
    g = run_gpu(soap, wl)
    assert g["info"]["n_visible"] == 70688
    assert g["n_active"].max() == 1920 and int(g["n_active"].sum()) == 20650
    for lo, hi in _sample_ranges(wl.n_pix):
        assert_parity(wl, g, lo, hi)


def test_config3_nested_variant_sampled(soap):
    wl = workloads.make_config3(nested=True)
    g = run_gpu(soap, wl)
    assert g["n_active"].max() == 1825 and int(g["n_active"].sum()) == 14694
    for lo, hi in _sample_ranges(wl.n_pix, n=3):
        assert_parity(wl, g, lo, hi)


def test_config4_full_size_sampled(soap):
    wl = workloads.make_config4()
    g = run_gpu(soap, wl)
    assert g["info"]["n_visible"] == 125676
    for lo, hi in _sample_ranges(wl.n_pix, width=512, n=2):
        assert_parity(wl, g, lo, hi)


def test_config5_batch_sampled(soap):
    """64 stars through the batch entry points; 3 stars x 2 ranges are checked against the oracle."""
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
    Q = torch.empty((n_stars, n_pix), dtype=torch.float32, device=dev)
    D = torch.empty((n_stars, n_ph, n_pix), dtype=torch.float32, device=dev)
    soap.soap_batch_integrate_quiet(stars, [q] * n_stars, [Q[k] for k in range(n_stars)])
    soap.soap_batch_active_timeseries(stars, [q] * n_stars, [s] * n_stars, [f] * n_stars, [w.regions for w in wls],
                                      [w.phases for w in wls], [D[k] for k in range(n_stars)])
    torch.cuda.synchronize()
    fastest = int(np.argmax([w.vsini_kms for w in wls]))
    for k in sorted({0, fastest, 63}):
        g = dict(Q=Q[k].cpu().numpy(), D=D[k].cpu().numpy(), n_active=None)
        wl = wls[k]
        for lo, hi in [(0, 512), (123_456, 123_456 + 512)]:
            Qo, Do, nao = oracle.run_workload(wl, lo, hi)
            sw = oracle.geometry(wl)["sum_w"]
            assert check_quiet(g["Q"][lo:hi], Qo, sw) <= QUIET_TOL
            if np.abs(Do).max() > 0:
                assert check_delta(g["D"][:, lo:hi], Do) <= DELTA_TOL
            else:
                assert np.all(g["D"][:, lo:hi] == 0.0)
            rv, _ = max_rv_diff(g["Q"][lo:hi].astype(np.float64), Qo, sw, wl, lo)
            assert rv <= RV_TOL_CMS
    for st in stars:
        soap.soap_destroy(st)


def test_batch_entry_points_equal_per_star_calls(soap):
    """soap_batch_* enqueue O(1) launches for the whole batch; every star's result equals the one its own calls give:
    to the last bit for the delta spectra (an item's result does not depend on which CTA computes it), and to an fp32
    rounding for the quiet spectra (the fp64 partial sums of a tile are grouped by CTA range, which depends on the batch)."""
    dev = torch.device("cuda:0")
    n_stars, n_pix, n_ph = 7, 30_000, 6
    shared = workloads.make_config5_star(0, n_pix=n_pix, n_phases=n_ph, grid_n=90)
    wls = [shared] + [workloads.make_config5_star(k, n_pix=n_pix, n_phases=n_ph, grid_n=90, shared=shared) for k in range(1, n_stars)]
    wls[2].regions = []                       # a star without regions: exact zeros
    wls[3].grid_n = 61                        # another grid: other column pairs, other tables
    q = soap.to_device_spectra(shared.quiet, shared.lambda0, shared.dlambda, dev)
    s = soap.to_device_spectra(shared.spot, shared.lambda0, shared.dlambda, dev, shared.spot_contrast, shared.spot_lb)
    f = soap.to_device_spectra(shared.facula, shared.lambda0, shared.dlambda, dev, shared.facula_contrast, shared.facula_lb)
    stars = [soap.soap_create(0) for _ in range(n_stars)]
    launches0 = sum(soap.soap_get_stats(st)["launches"] for st in stars)
    infos = soap.soap_batch_disk_geometry(stars, wls, want_info=True)
    for k, wl in enumerate(wls):              # one geometry launch for the batch: every star's cells as its own call gives them
        og = oracle.geometry(wl)
        assert infos[k]["n_visible"] == og["n_visible"] and abs(infos[k]["sum_weights"] - og["sum_w"]) <= 1e-9 * og["sum_w"]
    ref = soap.soap_create(0)
    soap.soap_disk_geometry(ref, wls[3], want_info=False)
    ga, gb = soap.soap_export_geometry(stars[3], wls[3].grid_n), soap.soap_export_geometry(ref, wls[3].grid_n)
    assert all(np.array_equal(ga[key], gb[key]) for key in ("mu", "w", "vel", "bin"))
    soap.soap_destroy(ref)
    Qb = torch.full((n_stars, n_pix), float("nan"), dtype=torch.float32, device=dev)
    Db = torch.full((n_stars, n_ph, n_pix), float("nan"), dtype=torch.float32, device=dev)
    soap.soap_batch_integrate_quiet(stars, [q] * n_stars, [Qb[k] for k in range(n_stars)])
    soap.soap_batch_active_timeseries(stars, [q] * n_stars, [s] * n_stars, [f] * n_stars, [w.regions for w in wls],
                                      [w.phases for w in wls], [Db[k] for k in range(n_stars)])
    torch.cuda.synchronize()
    launches = sum(soap.soap_get_stats(st)["launches"] for st in stars) - launches0
    assert launches <= 5, f"{launches} launches for {n_stars} stars: the batch entry points must not launch per star"
    assert not torch.isnan(Qb).any() and not torch.isnan(Db).any()
    for k, (st, wl) in enumerate(zip(stars, wls)):
        Q1 = torch.empty(n_pix, dtype=torch.float32, device=dev)
        D1 = torch.empty((n_ph, n_pix), dtype=torch.float32, device=dev)
        soap.soap_integrate_quiet(st, q, Q1)
        soap.soap_active_timeseries(st, q, s, f, wl.regions, wl.phases, D1)
        torch.cuda.synchronize()
        sw = oracle.geometry(wl)["sum_w"]
        assert float((Q1 - Qb[k]).abs().max()) <= 2.5e-7 * sw, f"star {k}"   # an fp32 ulp at the continuum level is 6e-8
        assert torch.equal(D1, Db[k]), f"star {k}"
        if not wl.regions:
            assert torch.all(Db[k] == 0.0)
    # and against the oracle for two of them
    for k in (1, 3):
        g = dict(Q=Qb[k].cpu().numpy(), D=Db[k].cpu().numpy(), n_active=oracle.run_workload(wls[k], 0, 16)[2])
        assert_parity(wls[k], g)
    for st in stars:
        soap.soap_destroy(st)


def test_host_buffer_entry_point(soap):
    wl = workloads.make_config2(n_pix=4000, n_phases=5, grid_n=80)
    wl.phases = np.linspace(0.35, 0.65, 5)
    star = soap.soap_create(0)
    pitch = (wl.n_pix + 3) & ~3

    def host(rows):
        t = torch.zeros((rows.shape[0], pitch), dtype=torch.float32).pin_memory()
        t[:, :wl.n_pix] = torch.from_numpy(rows)
        return t

    q = soap.Spectra(host(wl.quiet), wl.n_pix, wl.lambda0, wl.dlambda)
    s = soap.Spectra(host(wl.spot), wl.n_pix, wl.lambda0, wl.dlambda,
                     contrast=torch.from_numpy(wl.spot_contrast).pin_memory(), lb=wl.spot_lb)
    Q = torch.empty(wl.n_pix, dtype=torch.float32).pin_memory()
    D = torch.empty((len(wl.phases), wl.n_pix), dtype=torch.float32).pin_memory()
    na = soap.soap_synthesize_host(star, wl, q, s, None, wl.regions, wl.phases, Q, D, want_n_active=True)
    soap.soap_destroy(star)
    assert_parity(wl, dict(Q=Q.numpy(), D=D.numpy(), n_active=na))


def test_argument_errors_leave_outputs_untouched(soap):
    b = soap.binding
    wl = workloads.make_config2(n_pix=1000, n_phases=2, grid_n=30)
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    out = torch.full((wl.n_pix,), -7.0, dtype=torch.float32, device=dev)
    with pytest.raises(soap.SoapError) as e:
        soap.soap_integrate_quiet(star, q, out)
    assert e.value.code == b.SOAP_ERR_NOT_READY
    soap.soap_disk_geometry(star, wl)
    bad = soap.Spectra(q.data, q.n_pix, -1.0, q.dlambda)
    with pytest.raises(soap.SoapError) as e:
        soap.soap_integrate_quiet(star, bad, out)
    assert e.value.code == b.SOAP_ERR_INVALID_ARG
    D = torch.full((2, wl.n_pix), -7.0, dtype=torch.float32, device=dev)
    with pytest.raises(soap.SoapError) as e:  # a spot region without spot spectra
        soap.soap_active_timeseries(star, q, None, None, [(0.0, 180.0, 0.1, 1)], wl.phases, D)
    assert e.value.code == b.SOAP_ERR_INVALID_ARG
    with pytest.raises(soap.SoapError):
        soap.soap_active_timeseries(star, q, q, None, [(0.0, 180.0, 1.5, 1)], wl.phases, D)
    torch.cuda.synchronize()
    assert torch.all(out == -7.0) and torch.all(D == -7.0)
    soap.soap_destroy(star)


# ---- flux-only and CB-only outputs beside the total (Eq. 1-3) -------------------
def _run_effects(soap, wl, which=(True, True, True), passes=False, form=None):
    """`passes`: one shift-interpolate-accumulate pass per requested effect instead of one pass for all of them."""
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    if passes:
        soap.soap_set_option(star, soap.binding.SOAP_OPT_EFFECT_PASSES, 1)
    if form is not None:
        soap.soap_set_option(star, soap.binding.SOAP_OPT_FORM, form)
    soap.soap_disk_geometry(star, wl)
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    s = None if wl.spot is None else soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    f = None if wl.facula is None else soap.to_device_spectra(wl.facula, wl.lambda0, wl.dlambda, dev, wl.facula_contrast, wl.facula_lb)
    tdt = torch.float32 if wl.dtype == np.float32 else torch.float64
    outs = [torch.full((len(wl.phases), wl.n_pix), float("nan"), dtype=tdt, device=dev) if w else None for w in which]
    na = soap.soap_active_timeseries_effects(star, q, s, f, wl.regions, wl.phases, outs[0], outs[1], outs[2], want_n_active=True)
    torch.cuda.synchronize()
    soap.soap_destroy(star)
    return [o.cpu().numpy() if o is not None else None for o in outs], na


def _check_effects(wl, outs, na, m_lo=0, m_hi=None):
    scale = None
    for effect, D in enumerate(outs):
        if D is None:
            continue
        _, Do, nao = oracle.run_workload(wl, m_lo, m_hi, effect=effect)
        assert np.array_equal(na, nao)
        if scale is None:
            scale = float(np.max(np.abs(oracle.run_workload(wl, m_lo, m_hi, effect=0)[1])))
        # every effect is held to 1e-4 of its own max|delta|, and never looser than 1e-4 of the total's
        tol = DELTA_TOL * min(float(np.max(np.abs(Do))), scale) if np.max(np.abs(Do)) > 0 else 0.0
        err = float(np.max(np.abs(D[:, m_lo:m_hi].astype(np.float64) - Do)))
        assert err <= tol, f"effect {effect}: {err:.3e} > {tol:.3e}"
        for p in range(len(wl.phases)):
            if nao[p] == 0:
                assert np.all(D[p] == 0.0)


def test_effects_match_oracle_fp32(soap):
    wl = workloads.make_config3(n_pix=5000, n_phases=6, grid_n=120, nested=True)
    wl.phases = np.array([0.35, 0.45, 0.5, 0.55, 0.65, 0.0])
    outs, na = _run_effects(soap, wl)
    assert na.max() > 0
    _check_effects(wl, outs, na)


def test_effects_match_oracle_fp64_config1(soap):
    wl = workloads.make_config1()
    outs, na = _run_effects(soap, wl)
    _check_effects(wl, outs, na)


def test_effects_subsets_and_total_is_unchanged(soap):
    """Any subset of the outputs may be requested; with one pass per effect the total equals soap_active_timeseries bit
    for bit, and a single requested effect is that same pass."""
    wl = workloads.make_config2(n_pix=4000, n_phases=5, grid_n=100)
    wl.phases = np.linspace(0.4, 0.6, 5)
    g = run_gpu(soap, wl)
    (t, f, c), na = _run_effects(soap, wl, passes=True)
    assert np.array_equal(t, g["D"]) and np.array_equal(na, g["n_active"])
    (t2, f2, c2), _ = _run_effects(soap, wl, which=(False, True, False))
    assert t2 is None and c2 is None and np.array_equal(f2, f)
    (t3, f3, c3), _ = _run_effects(soap, wl, which=(False, False, True))
    assert np.array_equal(c3, c)
    _check_effects(wl, (t, f, c), na)


def _two_type_workload(lb):
    """A spot and a facula that overlap (columns and mu bins that hold cells of both types), second facula apart."""
    wl = workloads.make_config3(n_pix=5000, n_phases=5, grid_n=120, nested=True)
    wl.phases = np.array([0.42, 0.5, 0.58, 0.75, 0.0])
    wl.regions = list(wl.regions) + [(-20.0, 200.0, 0.12, 1)]
    wl.facula_contrast = (1.0 + 0.05 * np.sin(np.arange(wl.n_pix) / 50.0)).astype(np.float32)
    wl.spot_lb = (0.9, 0.1, 0.0) if lb == "both" else (1.0, 0.0, 0.0)
    wl.facula_lb = (1.1, -0.1, 0.0) if lb != "one" else (1.0, 0.0, 0.0)
    return wl


@pytest.mark.parametrize("lb", ["one", "facula", "both"])
def test_effects_one_pass_against_oracle_and_against_a_pass_per_effect(soap, lb):
    """Two or three requested effects come from ONE pass (entry lists of 4 kinds when both limb-brightening laws are 1;
    a type with a law gets two more): each against the oracle, and against the pass-per-effect form to a tenth of the
    parity tolerance."""
    wl = _two_type_workload(lb)
    assert {r[3] for r in wl.regions} == {1, 2}, "the workload must hold both region types"
    one, na = _run_effects(soap, wl)
    per, na2 = _run_effects(soap, wl, passes=True)
    assert np.array_equal(na, na2) and na.max() > 0
    _check_effects(wl, one, na)
    for a, b in zip(one, per):
        assert np.max(np.abs(a.astype(np.float64) - b)) <= 0.1 * DELTA_TOL * np.max(np.abs(b))
    again, _ = _run_effects(soap, wl)
    assert all(np.array_equal(a, b) for a, b in zip(one, again)), "the one-pass launch is run-to-run identical"
    # two of the three: the same pass with one output left out
    (t, f, c), _ = _run_effects(soap, wl, which=(True, False, True))
    assert f is None and np.array_equal(t, one[0]) and np.array_equal(c, one[2])
    (t, f, c), _ = _run_effects(soap, wl, which=(False, True, True))
    assert t is None and np.array_equal(f, one[1]) and np.array_equal(c, one[2])


def test_effects_config3_full_size_sampled(soap):
    wl = workloads.make_config3()
    outs, na = _run_effects(soap, wl)
    for lo, hi in _sample_ranges(wl.n_pix, n=2):
        _check_effects(wl, outs, na, lo, hi)


@pytest.mark.parametrize("form", [1, 3], ids=["binned", "fir"])
def test_effects_one_pass_in_the_binned_and_the_run_collapsed_form(soap, form):
    """The one-pass effects launch under SOAP_FORM_BINNED / SOAP_FORM_FIR (the active launch collapses runs of entries)."""
    wl = _two_type_workload("facula")
    wl.vsini_kms = 9.0
    outs, na = _run_effects(soap, wl, form=form)
    _check_effects(wl, outs, na)


def test_fir_form_config3_full_size_sampled(soap):
    """SOAP_FORM_FIR (every run of entries with one integer shift collapsed into one record) at full size."""
    wl = workloads.make_config3()
    g = run_gpu(soap, wl, form=3)
    assert g["stats"]["form"] == 3
    for lo, hi in _sample_ranges(wl.n_pix, n=3):
        assert_parity(wl, g, lo, hi)


def test_fir_form_fast_rotator(soap):
    wl = workloads.make_config5_star(3, n_pix=6000, n_phases=4, grid_n=90)
    wl.vsini_kms = 20.0
    wl.phases = np.array([0.4, 0.5, 0.6, 0.0])
    g = run_gpu(soap, wl, form=3)
    assert_parity(wl, g)


def test_host_buffer_entry_point_pipelined_chunks(soap):
    """Long fp32 spectra go through the chunked, three-stream host path: check chunk interiors, chunk boundaries and ends."""
    wl = workloads.make_config2(n_pix=150_000, n_phases=3, grid_n=40)
    wl.phases = np.array([0.45, 0.5, 0.0])
    wl.vsini_kms = 12.0
    star = soap.soap_create(0)
    pitch = (wl.n_pix + 3) & ~3

    def host(rows):
        t = torch.zeros((rows.shape[0], pitch), dtype=torch.float32).pin_memory()
        t[:, :wl.n_pix] = torch.from_numpy(rows)
        return t

    q = soap.Spectra(host(wl.quiet), wl.n_pix, wl.lambda0, wl.dlambda)
    s = soap.Spectra(host(wl.spot), wl.n_pix, wl.lambda0, wl.dlambda,
                     contrast=torch.from_numpy(wl.spot_contrast).pin_memory(), lb=wl.spot_lb)
    Q = torch.full((wl.n_pix,), float("nan"), dtype=torch.float32).pin_memory()
    D = torch.full((len(wl.phases), wl.n_pix), float("nan"), dtype=torch.float32).pin_memory()
    for _ in range(2):  # twice: buffers and events are reused
        na = soap.soap_synthesize_host(star, wl, q, s, None, wl.regions, wl.phases, Q, D, want_n_active=True)
    soap.soap_destroy(star)
    g = dict(Q=Q.numpy(), D=D.numpy(), n_active=na)
    assert not np.isnan(g["Q"]).any() and not np.isnan(g["D"]).any()
    tiles = (wl.n_pix + 2047) // 2048
    lc = ((tiles + 1) // 2) * 2048   # 74 tiles -> 2 chunks of 37 tiles
    for lo in (0, lc - 600, lc - 100, wl.n_pix - 900):
        assert_parity(wl, g, lo, lo + 900, check_rv=False)
    # against the device-resident path
    gd = run_gpu(soap, wl)
    assert np.max(np.abs(gd["Q"] - g["Q"])) <= 1e-6 * oracle.geometry(wl)["sum_w"]   # a few fp32 ulps
    assert np.max(np.abs(gd["D"] - g["D"])) <= 1e-5 * np.max(np.abs(gd["D"]))


def test_host_buffer_entry_point_pageable_buffers_and_bad_arguments(soap):
    """The chunked host path with ordinary (pageable) numpy-backed tensors for inputs and outputs: results are staged on the
    device and copied back chunk by chunk.  A bad table is refused before anything is enqueued: the outputs stay untouched."""
    wl = workloads.make_config2(n_pix=140_000, n_phases=3, grid_n=40)
    wl.phases = np.array([0.45, 0.5, 0.0])
    wl.vsini_kms = 8.0
    star = soap.soap_create(0)
    pitch = (wl.n_pix + 3) & ~3

    def host(rows):
        t = torch.zeros((rows.shape[0], pitch), dtype=torch.float32)
        t[:, :wl.n_pix] = torch.from_numpy(rows)
        return t

    q = soap.Spectra(host(wl.quiet), wl.n_pix, wl.lambda0, wl.dlambda)
    s = soap.Spectra(host(wl.spot), wl.n_pix, wl.lambda0, wl.dlambda, contrast=torch.from_numpy(wl.spot_contrast.copy()), lb=wl.spot_lb)
    Q = torch.full((wl.n_pix,), -7.0, dtype=torch.float32)
    D = torch.full((len(wl.phases), wl.n_pix), -7.0, dtype=torch.float32)
    assert not Q.is_pinned() and not D.is_pinned()
    bad = soap.Spectra(s.data, wl.n_pix, wl.lambda0, wl.dlambda, contrast=s.contrast, lb=(float("nan"), 0.0, 0.0))
    with pytest.raises(soap.SoapError) as e:
        soap.soap_synthesize_host(star, wl, q, bad, None, wl.regions, wl.phases, Q, D)
    assert e.value.code == soap.binding.SOAP_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert torch.all(Q == -7.0) and torch.all(D == -7.0)
    na = soap.soap_synthesize_host(star, wl, q, s, None, wl.regions, wl.phases, Q, D, want_n_active=True)
    soap.soap_destroy(star)
    g = dict(Q=Q.numpy(), D=D.numpy(), n_active=na)
    for lo in (0, 69_000, wl.n_pix - 900):
        assert_parity(wl, g, lo, lo + 900, check_rv=False)
