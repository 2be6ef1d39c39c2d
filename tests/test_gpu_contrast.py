"""SOAPcontrast on the device against the oracle's closed form.  -m gpu."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


@pytest.mark.parametrize("lambda0,k,n,tq,ta", [
    (3800.0, 0.01, 310_000, 5778.0, 4700.0),    # C3's grid, spot of BASELINE.json configs[1..2]
    (4500.0, 0.01, 200_000, 4500.0, 3500.0),    # C4: cool K dwarf
    (3800.0, 0.01, 310_000, 5778.0, 6028.9),    # a facula, hotter than the photosphere
    (500.0, 0.5, 4099, 5778.0, 4700.0),         # Wien regime (x ~ 50), ragged size
    (1e7, 1e5, 33, 5778.0, 4700.0),             # Rayleigh-Jeans regime
    (5293.0, 0.01, 1, 5778.0, 5115.0),          # the single value SOAP 2.0 used
])
def test_contrast_matches_oracle(soap, lambda0, k, n, tq, ta):
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    ref = oracle.contrast_planck(lambda0, k, n, tq, ta)
    o64 = torch.full((n,), float("nan"), dtype=torch.float64, device=dev)
    o32 = torch.full((n + 3,), float("nan"), dtype=torch.float32, device=dev)
    soap.soap_contrast_planck(star, lambda0, k, n, tq, ta, o64)
    soap.soap_contrast_planck(star, lambda0, k, n, tq, ta, o32)
    torch.cuda.synchronize()
    soap.soap_destroy(star)
    g64, g32 = o64.cpu().numpy(), o32.cpu().numpy()
    assert np.max(np.abs(g64 / ref - 1.0)) <= 1e-13
    assert np.max(np.abs(g32[:n].astype(np.float64) / ref - 1.0)) <= 1e-6     # north-star-style bar; an fp32 rounding is 6e-8
    assert np.max(np.abs(g32[:n].astype(np.float64) / ref - 1.0)) <= 6.1e-8
    assert np.all(np.isnan(g32[n:])), "nothing is written past n_pix"


def test_device_contrast_feeds_the_time_series(soap):
    """The kernel's output is what soap_spectra.contrast expects: the C2 time series computed with a contrast array made
    on the device equals (to fp32 rounding of the contrast) the one computed with the input generator's array."""
    dev = torch.device("cuda:0")
    wl = workloads.make_config2(n_pix=6000, n_phases=4, grid_n=80)
    wl.phases = np.array([0.45, 0.5, 0.55, 0.0])
    star = soap.soap_create(0)
    soap.soap_disk_geometry(star, wl)
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    s_ref = soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    c_dev = torch.empty(wl.n_pix, dtype=torch.float32, device=dev)
    soap.soap_contrast_planck(star, wl.lambda0, wl.dlambda, wl.n_pix, 5778.0, 4700.0, c_dev)
    s_dev = soap.Spectra(s_ref.data, wl.n_pix, wl.lambda0, wl.dlambda, contrast=c_dev, lb=wl.spot_lb)
    D1 = torch.empty((4, wl.n_pix), dtype=torch.float32, device=dev)
    D2 = torch.empty_like(D1)
    soap.soap_active_timeseries(star, q, s_ref, None, wl.regions, wl.phases, D1)
    soap.soap_active_timeseries(star, q, s_dev, None, wl.regions, wl.phases, D2)
    torch.cuda.synchronize()
    soap.soap_destroy(star)
    wl.spot_contrast = c_dev.cpu().numpy()
    Do = oracle.run_workload(wl)[1]
    assert float((D1 - D2).abs().max()) <= 2e-6 * float(D1.abs().max())
    assert np.max(np.abs(D2.cpu().numpy() - Do)) <= 1e-4 * np.max(np.abs(Do))


def test_contrast_argument_errors(soap):
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    out = torch.full((16,), -7.0, dtype=torch.float32, device=dev)
    for args in [(5000.0, 0.01, 16, 0.0, 4700.0), (5000.0, 0.01, 16, 5778.0, float("nan")), (-1.0, 0.01, 16, 5778.0, 4700.0),
                 (5000.0, 0.0, 16, 5778.0, 4700.0)]:
        with pytest.raises(soap.SoapError) as e:
            soap.soap_contrast_planck(star, *args, out)
        assert e.value.code == soap.binding.SOAP_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert torch.all(out == -7.0)
    soap.soap_destroy(star)
