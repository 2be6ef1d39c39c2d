"""soap_integrate_quiet_static: the quiet spectrum for callers that must not allocate device memory.  Needs a B200: -m gpu.

Who needs it: a program that has given the whole device to its own memory pool (a cudaMalloc made by this library would
fail there), or a service loop that cannot take the device-wide stall a cudaMalloc / cudaFree causes.  For them the entry
point keeps its fp64 partial sums in a fixed 4 MiB array inside the library instead of a buffer the handle grows on
demand (include/soap_b200.h states the limit, round_up4(n_pix) <= 524 288, and that overlapping calls race on the array).

What is checked, against the library's existing path (soap_integrate_quiet) on the same handle and tables, at the
tolerance the parity tests use for the quiet spectrum (helpers.QUIET_TOL of the integrated continuum):
  * two calls in a row on different tables - and of different lengths - each give the existing path's spectrum: the second
    call finds the first one's partial sums in the shared array and must not be affected by them;
  * fp64 tables, where both paths run the same kernels on the same chunks, agree bit for bit;
  * a spectrum exactly at the limit works, one past it is refused with a message that names the limit, output untouched.
The array lives as long as the process does, so nothing here depends on which tests ran before: this file is named to be
collected last only so that a failure in it cannot hide one elsewhere under `pytest -x`.
"""
from __future__ import annotations

import dataclasses

import numpy as np
import pytest

import workloads
from helpers import QUIET_TOL

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

STATIC_LIMIT_PX = 512 * 1024  # kStaticPartialDoubles in csrc/soap_api.cu


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


def _both_paths(soap, star, wl, rows):
    """Quiet spectrum of `rows` ([n_mu, P] numpy) through the existing entry point and through the static-scratch one."""
    dev = torch.device("cuda:0")
    q = soap.to_device_spectra(rows, wl.lambda0, wl.dlambda, dev)
    tdt = torch.float32 if rows.dtype == np.float32 else torch.float64
    ref = torch.full((rows.shape[1],), float("nan"), dtype=tdt, device=dev)
    got = torch.full((rows.shape[1],), float("nan"), dtype=tdt, device=dev)
    soap.soap_integrate_quiet(star, q, ref)
    soap.soap_integrate_quiet_static(star, q, got)
    torch.cuda.synchronize()
    return ref.cpu().numpy().astype(np.float64), got.cpu().numpy().astype(np.float64)


def _assert_same(ref, got, sum_w, what):
    assert np.all(np.isfinite(got)), f"{what}: static-scratch path left pixels unwritten"
    err = float(np.max(np.abs(got - ref))) / sum_w
    assert err <= QUIET_TOL, f"{what}: differs from soap_integrate_quiet by {err:.3e} of the continuum"
    return err


def test_fp32_two_calls_in_a_row_match_the_existing_path(soap):
    wl = workloads.make_config2(n_pix=10_000, n_phases=1)  # N=300, 20 mu bins, fp32
    star = soap.soap_create(0)
    try:
        info = soap.soap_disk_geometry(star, wl)
        sw = info["sum_weights"]
        # call 1: the table as generated
        ref1, got1 = _both_paths(soap, star, wl, wl.quiet)
        _assert_same(ref1, got1, sw, "first call")
        # call 2, straight after: a different and shorter table (reversed bins, scaled, ragged length) - the array still holds
        # call 1's partial sums beyond and inside the part this call uses
        rows2 = np.ascontiguousarray((0.5 * wl.quiet[::-1, :4099]).astype(np.float32))
        ref2, got2 = _both_paths(soap, star, wl, rows2)
        _assert_same(ref2, got2, sw, "second call")
        assert float(np.max(np.abs(ref2 - ref1[:4099]))) > 1e-3 * sw  # the two calls really had different answers
        # and the first table once more: same bits as before (the path is run-to-run identical)
        _, got3 = _both_paths(soap, star, wl, wl.quiet)
        assert np.array_equal(got3, got1)
    finally:
        soap.soap_destroy(star)


def test_fp64_two_calls_in_a_row_are_bit_identical_to_the_existing_path(soap):
    wl = workloads.make_config1()  # N=50, 2000 px, one mu bin, fp64
    star = soap.soap_create(0)
    try:
        info = soap.soap_disk_geometry(star, wl)
        sw = info["sum_weights"]
        ref1, got1 = _both_paths(soap, star, wl, wl.quiet)
        _assert_same(ref1, got1, sw, "first call")
        assert np.array_equal(ref1, got1)
        rows2 = np.ascontiguousarray(1.0 - 0.25 * wl.quiet[:, :1501])
        ref2, got2 = _both_paths(soap, star, wl, rows2)
        _assert_same(ref2, got2, sw, "second call")
        assert np.array_equal(ref2, got2)
    finally:
        soap.soap_destroy(star)


def test_limit_of_the_static_scratch(soap):
    base = workloads.make_config1()
    rng = np.random.default_rng(workloads.SEED_BASE + 77)
    star = soap.soap_create(0)
    try:
        info = soap.soap_disk_geometry(star, base)
        sw = info["sum_weights"]
        # exactly at the limit: one chunk of entries, the whole array in use
        rows = 1.0 - 0.5 * rng.random((1, STATIC_LIMIT_PX))
        wl = dataclasses.replace(base, n_pix=STATIC_LIMIT_PX, quiet=rows)
        ref, got = _both_paths(soap, star, wl, rows)
        _assert_same(ref, got, sw, "n_pix at the limit")
        # one quad past it: refused, message names the limit, output untouched
        dev = torch.device("cuda:0")
        rows_big = np.ones((1, STATIC_LIMIT_PX + 1))
        q = soap.to_device_spectra(rows_big, base.lambda0, base.dlambda, dev)
        out = torch.full((STATIC_LIMIT_PX + 1,), float("nan"), dtype=torch.float64, device=dev)
        with pytest.raises(soap.SoapError) as ei:
            soap.soap_integrate_quiet_static(star, q, out)
        assert ei.value.code == soap.binding.SOAP_ERR_UNSUPPORTED
        assert "static scratch" in str(ei.value) and str(STATIC_LIMIT_PX) in str(ei.value)
        torch.cuda.synchronize()
        assert bool(torch.isnan(out).all())
        # the same table through the allocating entry point is fine
        soap.soap_integrate_quiet(star, q, out)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(out).all())
    finally:
        soap.soap_destroy(star)


def test_needs_geometry_first(soap):
    wl = workloads.make_config1()
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    try:
        q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
        out = torch.zeros((wl.n_pix,), dtype=torch.float64, device=dev)
        with pytest.raises(soap.SoapError) as ei:
            soap.soap_integrate_quiet_static(star, q, out)
        assert ei.value.code == soap.binding.SOAP_ERR_NOT_READY
    finally:
        soap.soap_destroy(star)
