"""Cases found in review that no other test reached (needs a B200: -m gpu).

  * one handle re-used back to back: the launches of consecutive calls are chained with programmatic dependent launch, so a
    call's kernels may be resident while the previous call's are still draining; what one call's map / geometry launch
    wrote must be what the next launch reads (those buffers are read with ld.global.cg, never through the read-only path);
  * a batch whose stars each fit the one-launch composite form but not together (fine grid + fast rotator);
  * differential rotation with fp32 tables on a grid whose binned active map would not fit in shared memory - the per-cell
    map that this path uses does.
"""
from __future__ import annotations

import dataclasses

import numpy as np
import pytest

import oracle
import workloads
from helpers import QUIET_TOL, check_quiet
from test_gpu_parity import assert_parity, run_gpu

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


def test_consecutive_calls_on_one_handle_equal_fresh_handles(soap):
    """geometry -> quiet -> series -> series -> geometry -> quiet -> series on ONE handle with nothing but the stream between
    them, each step with other regions / phases / star parameters: every output equals, bit for bit, what a fresh handle
    gives for the same inputs."""
    dev = torch.device("cuda:0")
    n_pix = 20_000
    wl_a = workloads.make_config3(n_pix=n_pix, n_phases=6, grid_n=300)
    wl_b = dataclasses.replace(wl_a, regions=[(35.0, 150.0, 0.22, 2), (-10.0, 200.0, 0.12, 1), (5.0, 170.0, 0.05, 2)],
                               phases=np.array([0.52, 0.04, 0.47, 0.4, 0.6, 0.55, 0.5, 0.45, 0.35]))
    wl_c = dataclasses.replace(wl_a, grid_n=257, vsini_kms=7.5, incl_deg=70.0, regions=[(20.0, 185.0, 0.3, 1)],
                               phases=np.array([0.5, 0.45, 0.55]))
    refs = [run_gpu(soap, w, want_n_active=False) for w in (wl_a, wl_b, wl_c)]
    q = soap.to_device_spectra(wl_a.quiet, wl_a.lambda0, wl_a.dlambda, dev)
    s = soap.to_device_spectra(wl_a.spot, wl_a.lambda0, wl_a.dlambda, dev, wl_a.spot_contrast, wl_a.spot_lb)
    f = soap.to_device_spectra(wl_a.facula, wl_a.lambda0, wl_a.dlambda, dev, wl_a.facula_contrast, wl_a.facula_lb)
    for rep in range(3):  # (which CTAs overlap differs from run to run)
        star = soap.soap_create(0)
        Q = [torch.full((n_pix,), float("nan"), dtype=torch.float32, device=dev) for _ in range(2)]
        D = [torch.full((len(w.phases), n_pix), float("nan"), dtype=torch.float32, device=dev) for w in (wl_a, wl_b, wl_c)]
        soap.soap_disk_geometry(star, wl_a, want_info=False)
        soap.soap_integrate_quiet(star, q, Q[0])
        soap.soap_active_timeseries(star, q, s, f, wl_a.regions, wl_a.phases, D[0], want_n_active=False)
        soap.soap_active_timeseries(star, q, s, f, wl_b.regions, wl_b.phases, D[1], want_n_active=False)
        soap.soap_disk_geometry(star, wl_c, want_info=False)
        soap.soap_integrate_quiet(star, q, Q[1])
        soap.soap_active_timeseries(star, q, s, f, wl_c.regions, wl_c.phases, D[2], want_n_active=False)
        torch.cuda.synchronize()
        soap.soap_destroy(star)
        assert np.array_equal(Q[0].cpu().numpy(), refs[0]["Q"]) and np.array_equal(Q[1].cpu().numpy(), refs[2]["Q"]), rep
        for k in range(3):
            assert np.array_equal(D[k].cpu().numpy(), refs[k]["D"]), (rep, k)
    assert np.any(refs[1]["D"] != 0.0) and np.any(refs[2]["D"] != 0.0)


def test_batch_quiet_of_a_fine_grid_and_a_fast_rotator(soap):
    """Each star qualifies for the one-launch composite form; together the launch would need the fine grid's pair table and
    the fast rotator's halo at once, which does not fit: the batch call must fall back to per-star launches, not fail."""
    dev = torch.device("cuda:0")
    n_pix = 3000
    shared = workloads.make_config5_star(0, n_pix=n_pix, n_phases=2, grid_n=1200)
    fast = workloads.make_config5_star(1, n_pix=n_pix, n_phases=2, grid_n=60, shared=shared)
    shared.vsini_kms, shared.incl_deg = 2.0, 90.0
    fast.incl_deg = 90.0
    fast.vsini_kms = 420.0 / (fast.lambda0 / fast.dlambda + n_pix) * 299792.458  # limb shift of about 420 pixels
    wls = [shared, fast]
    q = soap.to_device_spectra(shared.quiet, shared.lambda0, shared.dlambda, dev)
    stars = [soap.soap_create(0) for _ in wls]
    infos = [soap.soap_disk_geometry(st, wl) for st, wl in zip(stars, wls)]
    shift = infos[1]["max_abs_dshift"] * (fast.lambda0 / fast.dlambda + n_pix)
    assert 340.0 < shift < 500.0 and infos[0]["n_visible"] > 1_000_000  # the combination this test is about
    Qb = torch.full((2, n_pix), float("nan"), dtype=torch.float32, device=dev)
    soap.soap_batch_integrate_quiet(stars, [q, q], [Qb[0], Qb[1]])
    torch.cuda.synchronize()
    for k, (st, wl) in enumerate(zip(stars, wls)):
        Q1 = torch.full((n_pix,), float("nan"), dtype=torch.float32, device=dev)
        soap.soap_integrate_quiet(st, q, Q1)
        torch.cuda.synchronize()
        assert soap.soap_get_stats(st)["form"] == soap.binding.SOAP_FORM_COMPOSITE
        assert float((Q1 - Qb[k]).abs().max()) <= 2.5e-7 * infos[k]["sum_weights"], f"star {k}"
    Qo, _, _ = oracle.run_workload(fast)
    assert check_quiet(Qb[1].cpu().numpy(), Qo, oracle.geometry(fast)["sum_w"]) <= QUIET_TOL
    for st in stars:
        soap.soap_destroy(st)


def test_diffrot_fp32_on_a_grid_too_large_for_the_binned_active_map(soap):
    """N = 1100 with 64 mu bins: the binned active-map kernel would need 3 x 64 x 138 fp64 sums (> 200 KB) per CTA, but under
    differential rotation the map is built per cell (int counters, half the size) and the launch that follows must not
    apply the binned kernel's limit."""
    base = workloads.make_config3(n_pix=640, n_phases=2, grid_n=1100)
    pick = np.arange(64) % base.n_mu
    wl = dataclasses.replace(base, mu_centres=(np.arange(64, dtype=np.float64) + 0.5) / 64.0,
                             quiet=np.ascontiguousarray(base.quiet[pick]), spot=np.ascontiguousarray(base.spot[pick]),
                             facula=np.ascontiguousarray(base.facula[pick]), diff_rot=-0.18, incl_deg=70.0,
                             phases=np.array([0.5, 0.3]))
    g = run_gpu(soap, wl)
    assert g["n_active"].max() > 0
    assert_parity(wl, g, check_rv=False)
