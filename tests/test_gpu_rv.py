"""Parity of soap_line_rvs (first-moment line RVs on the device) against the oracle; needs a B200: -m gpu."""
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


def _gpu(soap, rows, wl, half, norm, edge):
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    x = torch.from_numpy(np.ascontiguousarray(rows)).to(dev)
    out = soap.soap_line_rvs(star, x, wl.n_pix, wl.lambda0, wl.dlambda, torch.from_numpy(wl.line_centres.astype(np.float64)).to(dev),
                             torch.from_numpy(half.astype(np.float64)).to(dev),
                             torch.from_numpy(np.broadcast_to(np.float64(norm), (rows.shape[0],)).copy()).to(dev), edge)
    torch.cuda.synchronize()
    soap.soap_destroy(star)
    return out.cpu().numpy()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_line_rvs_match_oracle(soap, dtype):
    wl = workloads.make_config2(n_pix=8000, n_phases=3, grid_n=50)
    Q, D, _ = oracle.run_workload(wl)
    sw = oracle.geometry(wl)["sum_w"]
    rows = np.vstack([Q[None, :], Q[None, :] + D]).astype(dtype)
    half = 3.0 * np.maximum(wl.line_sigmas, 0.03)
    a = _gpu(soap, rows, wl, half, sw, 64)
    b = oracle.line_rvs(rows.astype(np.float64), wl.lambda0, wl.dlambda, wl.line_centres, half, sw, edge=64)
    assert np.array_equal(np.isnan(a), np.isnan(b)) and np.sum(~np.isnan(b)) > 500
    np.testing.assert_allclose(a[~np.isnan(a)], b[~np.isnan(b)], rtol=1e-9, atol=1e-5)   # 1e-5 cm/s


def test_line_rvs_full_size(soap):
    """25 000 lines x 26 rows of 310 000 px: a sample of lines against the oracle."""
    wl = workloads.make_config3()
    rows = np.vstack([wl.quiet, wl.spot[:6]]).astype(np.float32)[:26]
    half = 3.0 * np.maximum(wl.line_sigmas, 0.03)
    a = _gpu(soap, rows, wl, half, 1.0, 64)
    sel = np.random.default_rng(7).choice(len(wl.line_centres), 400, replace=False)
    b = oracle.line_rvs(rows.astype(np.float64), wl.lambda0, wl.dlambda, wl.line_centres[sel], half[sel], 1.0, edge=64)
    a = a[:, sel]
    assert np.array_equal(np.isnan(a), np.isnan(b))
    np.testing.assert_allclose(a[~np.isnan(a)], b[~np.isnan(b)], rtol=1e-9, atol=1e-5)
