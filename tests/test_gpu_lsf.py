"""Parity of soap_lower_resolution against the fp64 oracle; needs a B200: -m gpu."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import workloads
from helpers import QUIET_TOL, RV_TOL_CMS, max_rv_diff

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

R_HARPSN = 115000.0


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


def _lower(soap, rows, n_pix, lam0, k, R, pitch=None):
    dev = torch.device("cuda:0")
    rows = np.atleast_2d(rows)
    pitch = pitch or n_pix
    tdt = torch.float32 if rows.dtype == np.float32 else torch.float64
    x = torch.zeros((rows.shape[0], pitch), dtype=tdt, device=dev)
    x[:, :n_pix] = torch.from_numpy(rows).to(dev)
    y = torch.full((rows.shape[0], pitch), float("nan"), dtype=tdt, device=dev)
    star = soap.soap_create(0)
    soap.soap_lower_resolution(star, x, n_pix, lam0, k, R, y)
    torch.cuda.synchronize()
    soap.soap_destroy(star)
    return y.cpu().numpy()[:, :n_pix]


def test_lsf_fp64_matches_oracle_tightly(soap):
    wl = workloads.make_config1()
    F, D, _ = oracle.run_workload(wl)
    rows = np.vstack([F[None, :], F[None, :] + D])  # quiet and the final spectrum of every phase (Eq. 4)
    y = _lower(soap, rows, wl.n_pix, wl.lambda0, wl.dlambda, R_HARPSN)
    yo = oracle.lower_resolution(rows, wl.lambda0, wl.dlambda, R_HARPSN)
    np.testing.assert_allclose(y, yo, rtol=1e-13)


@pytest.mark.parametrize("n_pix", [1, 2, 7, 255, 256, 257, 1000, 4099])
def test_lsf_ragged_sizes_and_edges(soap, n_pix):
    rng = np.random.default_rng(n_pix)
    rows = rng.uniform(0.2, 1.0, (3, n_pix)).astype(np.float32)
    y = _lower(soap, rows, n_pix, 6800.0, 0.01, 60000.0, pitch=(n_pix + 3) & ~3)   # wide LSF: J ~ 25 px
    yo = oracle.lower_resolution(rows.astype(np.float64), 6800.0, 0.01, 60000.0)
    assert np.max(np.abs(y - yo)) <= 2e-7


def test_lsf_final_spectra_rv_parity(soap):
    """Q + delta_p of a line-window workload, lowered to R = 115 000: value and per-line RV parity."""
    wl = workloads.make_config2(n_pix=6000, n_phases=4, grid_n=60)
    wl.phases = np.array([0.4, 0.5, 0.6, 0.0])
    Q, D, _ = oracle.run_workload(wl)
    sw = oracle.geometry(wl)["sum_w"]
    rows = (Q[None, :] + D).astype(np.float32)          # what the library would hand over, rounded to its I/O type
    y = _lower(soap, rows, wl.n_pix, wl.lambda0, wl.dlambda, R_HARPSN)
    yo = oracle.lower_resolution(rows.astype(np.float64), wl.lambda0, wl.dlambda, R_HARPSN)
    assert np.max(np.abs(y - yo)) <= QUIET_TOL * sw
    rv, n = max_rv_diff(y.astype(np.float64), yo, sw, wl)
    assert n > 0 and rv <= RV_TOL_CMS, f"{rv:.3f} cm/s over {n} lines"


def test_lsf_full_size_rows(soap):
    """BASELINE configs[2] shape: 26 rows x 310 000 px (fp32), sampled against the oracle."""
    wl = workloads.make_config3()
    rows = np.vstack([wl.quiet, wl.spot[:6]]).astype(np.float32)[:26]
    y = _lower(soap, rows, wl.n_pix, wl.lambda0, wl.dlambda, R_HARPSN)
    for lo in (0, 150_000, wl.n_pix - 4096):
        hi = lo + 4096
        a, b = max(0, lo - 64), min(wl.n_pix, hi + 64)
        yo = oracle.lower_resolution(rows[:, a:b].astype(np.float64), wl.lambda0 + wl.dlambda * a, wl.dlambda, R_HARPSN)
        sl = slice(lo - a, lo - a + 4096)
        if lo == 0:
            assert np.max(np.abs(y[:, :4096] - yo[:, :4096])) <= 2e-7
        elif hi == wl.n_pix:
            assert np.max(np.abs(y[:, lo:hi] - yo[:, sl])) <= 2e-7
        else:
            assert np.max(np.abs(y[:, lo:hi] - yo[:, sl])) <= 2e-7


def test_lsf_argument_errors(soap):
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    x = torch.ones((2, 100), dtype=torch.float32, device=dev)
    y = torch.full((2, 100), -7.0, dtype=torch.float32, device=dev)
    with pytest.raises(soap.SoapError):
        soap.soap_lower_resolution(star, x, 100, 5000.0, 0.01, -1.0, y)
    with pytest.raises(soap.SoapError):
        soap.soap_lower_resolution(star, x, 100, 5000.0, 0.01, 1000.0, y)   # LSF wider than the kernel supports
    with pytest.raises(soap.SoapError):
        soap.soap_lower_resolution(star, x, 100, 5000.0, 0.01, 1e5, x)
    torch.cuda.synchronize()
    assert torch.all(y == -7.0)
    soap.soap_destroy(star)
