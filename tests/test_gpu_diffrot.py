"""Parity of the per-cell path under differential rotation against the oracle."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import assert_parity, run_gpu, _sample_ranges

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


def test_diffrot_geometry_is_bit_exact(soap):
    wl = workloads.make_config2(n_pix=2000, n_phases=2, grid_n=150)
    wl.diff_rot, wl.incl_deg = -0.18, 60.0
    g = run_gpu(soap, wl)
    og = oracle.geometry(wl)
    np.testing.assert_array_equal(g["geo"]["vel"], og["vel"])
    np.testing.assert_array_equal(g["geo"]["bin"], og["bin"])
    assert g["stats"]["form"] == 3 and g["info"]["n_entries"] == og["n_visible"]  # AUTO: per-cell entries, runs collapsed


@pytest.mark.parametrize("dr,incl", [(-0.18, 90.0), (-0.18, 55.0), (0.25, 70.0)])
def test_diffrot_quiet_and_active_parity(soap, dr, incl):
    wl = workloads.make_config3(n_pix=6000, n_phases=6, grid_n=110, nested=True)
    wl.diff_rot, wl.incl_deg, wl.vsini_kms = dr, incl, 6.0
    wl.phases = np.array([0.35, 0.45, 0.5, 0.55, 0.65, 0.0])
    g = run_gpu(soap, wl)
    assert g["n_active"].max() > 0
    assert_parity(wl, g)


def test_diffrot_direct_per_cell_form(soap):
    """SOAP_FORM_CELLS under differential rotation: one lerp-accumulate per (cell, pixel), no run collapse."""
    wl = workloads.make_config3(n_pix=5000, n_phases=4, grid_n=90)
    wl.diff_rot, wl.incl_deg = -0.18, 65.0
    wl.phases = np.array([0.1, 0.2, 0.45, 0.55])
    g = run_gpu(soap, wl, form=2)
    assert g["stats"]["form"] == 2
    assert_parity(wl, g)


def test_diffrot_many_regions_and_limb(soap):
    wl = workloads.make_config4(n_pix=5000, n_phases=8, grid_n=90)
    wl.diff_rot = -0.2
    g = run_gpu(soap, wl)
    assert_parity(wl, g)


def test_diffrot_fir_form_and_effects(soap):
    wl = workloads.make_config3(n_pix=4000, n_phases=4, grid_n=80)
    wl.diff_rot, wl.incl_deg = -0.18, 75.0
    wl.phases = np.array([0.1, 0.2, 0.45, 0.55])
    g = run_gpu(soap, wl, form=3)
    assert_parity(wl, g)
    from test_gpu_parity import _run_effects, _check_effects
    outs, na = _run_effects(soap, wl)
    _check_effects(wl, outs, na)


def test_diffrot_full_size_config3_sampled(soap):
    wl = workloads.make_config3()
    wl.diff_rot = -0.18
    g = run_gpu(soap, wl)
    assert g["info"]["n_visible"] == 70688
    for lo, hi in _sample_ranges(wl.n_pix, n=2):
        assert_parity(wl, g, lo, hi)


def test_diffrot_rejects_binned_form_and_runs_fp64(soap):
    wl = workloads.make_config1()
    wl.diff_rot = -0.18
    star = soap.soap_create(0)
    soap.soap_set_option(star, soap.binding.SOAP_OPT_FORM, 1)
    with pytest.raises(soap.SoapError) as e:
        soap.soap_disk_geometry(star, wl)
    assert e.value.code == soap.binding.SOAP_ERR_UNSUPPORTED
    soap.soap_destroy(star)
    g = run_gpu(soap, wl)                                        # fp64 I/O: generic kernel, fixed-slot per-cell entries
    Qo, Do, nao = oracle.run_workload(wl)
    sw = oracle.geometry(wl)["sum_w"]
    assert np.max(np.abs(g["Q"] - Qo)) <= 1e-9 * sw
    assert np.array_equal(g["n_active"], nao) and nao.max() > 0
    assert np.max(np.abs(g["D"] - Do)) <= 1e-9 * np.max(np.abs(Do))
    assert_parity(wl, g)


def test_mixed_batch_with_a_differentially_rotating_star(soap):
    """soap_batch_* with one differentially rotating star among solid-body ones: one geometry launch for all (plus the star's
    per-cell entry launch), the quiet / active calls fall back to per-star launches; every star's result equals its own calls'."""
    dev = torch.device("cuda:0")
    n_pix, n_ph = 12_000, 4
    shared = workloads.make_config5_star(0, n_pix=n_pix, n_phases=n_ph, grid_n=70)
    wls = [shared] + [workloads.make_config5_star(k, n_pix=n_pix, n_phases=n_ph, grid_n=70, shared=shared) for k in (1, 2)]
    wls[1].diff_rot = -0.18
    q = soap.to_device_spectra(shared.quiet, shared.lambda0, shared.dlambda, dev)
    s = soap.to_device_spectra(shared.spot, shared.lambda0, shared.dlambda, dev, shared.spot_contrast, shared.spot_lb)
    f = soap.to_device_spectra(shared.facula, shared.lambda0, shared.dlambda, dev, shared.facula_contrast, shared.facula_lb)
    stars = [soap.soap_create(0) for _ in wls]
    soap.soap_batch_disk_geometry(stars, wls)
    Qb = torch.full((3, n_pix), float("nan"), dtype=torch.float32, device=dev)
    Db = torch.full((3, n_ph, n_pix), float("nan"), dtype=torch.float32, device=dev)
    soap.soap_batch_integrate_quiet(stars, [q] * 3, [Qb[k] for k in range(3)])
    soap.soap_batch_active_timeseries(stars, [q] * 3, [s] * 3, [f] * 3, [w.regions for w in wls], [w.phases for w in wls],
                                      [Db[k] for k in range(3)])
    torch.cuda.synchronize()
    for k, wl in enumerate(wls):
        ref = soap.soap_create(0)
        soap.soap_disk_geometry(ref, wl, want_info=False)
        Q1 = torch.empty(n_pix, dtype=torch.float32, device=dev)
        D1 = torch.empty((n_ph, n_pix), dtype=torch.float32, device=dev)
        soap.soap_integrate_quiet(ref, q, Q1)
        soap.soap_active_timeseries(ref, q, s, f, wl.regions, wl.phases, D1)
        torch.cuda.synchronize()
        assert torch.equal(Q1, Qb[k]) and torch.equal(D1, Db[k]), f"star {k}"
        soap.soap_destroy(ref)
    Qo, Do, _ = oracle.run_workload(wls[1])
    sw = oracle.geometry(wls[1])["sum_w"]
    assert float(np.max(np.abs(Qb[1].cpu().numpy() - Qo))) <= 1e-5 * sw
    assert float(np.max(np.abs(Db[1].cpu().numpy() - Do))) <= 1e-4 * float(np.max(np.abs(Do)))
    for st in stars:
        soap.soap_destroy(st)
