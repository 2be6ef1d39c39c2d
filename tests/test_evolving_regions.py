"""Evolving regions: a radius per (phase, region).

CPU part: the oracle wrapper is a plain loop over the pinned `oracle.active`; its own pins are the reductions to it.
GPU part (-m gpu): soap_active_timeseries_evolving against the oracle, incl. a many-region workload."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import workloads


def _wl(n_pix=1500, grid_n=50, n_phases=6):
    wl = workloads.make_config3(n_pix=n_pix, n_phases=n_phases, grid_n=grid_n)
    wl.vsini_kms = 6.0
    wl.regions = [(-20.0, 170.0, 0.2, 2), (15.0, 185.0, 0.12, 1)]
    wl.phases = np.linspace(0.42, 0.58, n_phases)
    return wl


def _orc(wl, radii, effect=0, m_lo=0, m_hi=None):
    return oracle.active_evolving(wl, wl.quiet, wl.spot, wl.facula, wl.lambda0, wl.dlambda, wl.regions, wl.phases, radii,
                                  wl.spot_contrast, wl.facula_contrast, wl.spot_lb, wl.facula_lb, m_lo, m_hi, effect)


def test_constant_radii_reduce_to_the_static_series_and_absent_regions_vanish():
    wl = _wl()
    const = np.tile([r[2] for r in wl.regions], (len(wl.phases), 1))
    D0, n0 = oracle.run_workload(wl)[1:]
    D1, n1 = _orc(wl, const)
    np.testing.assert_array_equal(D0, D1)
    np.testing.assert_array_equal(n0, n1)
    gone = const.copy()
    gone[2:4, :] = 0.0                       # both regions absent at phases 2, 3
    D2, n2 = _orc(wl, gone)
    assert np.all(D2[2:4] == 0.0) and list(n2[2:4]) == [0, 0]
    np.testing.assert_array_equal(D2[[0, 1, 4, 5]], D0[[0, 1, 4, 5]])


def test_growing_region_covers_more_cells_and_evolution_laws():
    wl = _wl()
    t = np.linspace(0.0, 10.0, len(wl.phases))
    grow = workloads.evolution_radii("growth", t)                        # 10 000 MSH + 400 MSH / day
    assert abs(grow[0] - 0.1) < 1e-15 and abs(grow[-1] - np.sqrt(0.014)) < 1e-15
    decay = workloads.evolution_radii("decay", np.array([0.0, 25.0, 30.0]))
    assert decay[1] == 0.0 and decay[2] == 0.0                           # 10 000 - 400 * 25 = 0
    gauss = workloads.evolution_radii("gaussian", np.array([-5.0, 0.0, 5.0]))
    assert gauss[1] == 0.1 and gauss[0] < gauss[2] < gauss[1]             # asymmetric: faster rise than decay
    wl.regions = [(0.0, 180.0, 0.1, 1)]
    wl.phases = np.full(len(t), 0.5)
    _, n = _orc(wl, grow[:, None])
    assert np.all(np.diff(n) >= 0) and n[-1] > n[0]


# ---- GPU parity ------------------------------------------------------------------------------------------------
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


def _gpu(soap, wl, radii, which=(True, False, False)):
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    soap.soap_disk_geometry(star, wl)
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    s = soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    f = soap.to_device_spectra(wl.facula, wl.lambda0, wl.dlambda, dev, wl.facula_contrast, wl.facula_lb)
    outs = [torch.full((len(wl.phases), wl.n_pix), float("nan"), dtype=torch.float32, device=dev) if w else None for w in which]
    na = soap.soap_active_timeseries_evolving(star, q, s, f, wl.regions, wl.phases, radii, outs[0], outs[1], outs[2], want_n_active=True)
    torch.cuda.synchronize()
    soap.soap_destroy(star)
    return [o.cpu().numpy() if o is not None else None for o in outs], na


@pytest.mark.gpu
@pytest.mark.parametrize("dr", [0.0, -0.18])
def test_gpu_evolving_regions_match_oracle(soap, dr):
    wl = _wl(n_pix=5000, grid_n=100, n_phases=8)
    wl.diff_rot = dr
    t = np.linspace(-6.0, 8.0, len(wl.phases))
    radii = np.stack([2.0 * workloads.evolution_radii("gaussian", t), workloads.evolution_radii("decay", t + 20.0)], axis=1)
    assert radii[:, 1].min() == 0.0 and radii[:, 1].max() > 0.0      # the spot dies during the series
    outs, na = _gpu(soap, wl, radii, which=(True, True, True))
    for effect in (0, 1, 2):
        Do, nao = _orc(wl, radii, effect)
        assert np.array_equal(na, nao)
        assert np.max(np.abs(outs[effect] - Do)) <= 1e-4 * np.max(np.abs(Do))
        for p in range(len(wl.phases)):
            if nao[p] == 0:
                assert np.all(outs[effect][p] == 0.0)


@pytest.mark.gpu
def test_gpu_hundreds_of_regions(soap):
    """P:426 'hundreds of active regions': 300 seeded regions, list-order override everywhere."""
    wl = _wl(n_pix=3000, grid_n=120, n_phases=5)
    rng = np.random.default_rng(426)
    wl.regions = [(float(rng.uniform(-70, 70)), float(rng.uniform(0, 360)), float(rng.uniform(0.02, 0.08)), int(rng.integers(1, 3)))
                  for _ in range(300)]
    wl.phases = np.array([0.0, 0.2, 0.4, 0.6, 0.8])
    radii = np.tile([r[2] for r in wl.regions], (5, 1))
    outs, na = _gpu(soap, wl, radii)
    Do, nao = oracle.run_workload(wl)[1:]
    assert np.array_equal(na, nao) and nao.min() > 1000
    assert np.max(np.abs(outs[0] - Do)) <= 1e-4 * np.max(np.abs(Do))
