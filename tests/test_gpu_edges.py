"""Degenerate and extreme inputs of the hot path against the oracle (needs a B200: -m gpu)."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
import workloads
from test_gpu_parity import assert_parity, run_gpu

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def soap():
    import paper_2301_04259_b200 as soap_mod
    soap_mod.binding.load_library()
    return soap_mod


@pytest.mark.parametrize("grid_n", [1, 2, 3, 7, 33])
def test_tiny_grids(soap, grid_n):
    wl = workloads.make_config2(n_pix=2500, n_phases=3, grid_n=grid_n)
    wl.regions = [(0.0, 180.0, 0.6, 1)]
    wl.phases = np.array([0.5, 0.25, 0.0])
    g = run_gpu(soap, wl)
    assert g["info"]["n_visible"] == oracle.geometry(wl)["n_visible"]
    assert_parity(wl, g, check_rv=False)


def test_one_mu_bin_and_sixty_four_mu_bins(soap):
    wl = workloads.make_config2(n_pix=3000, n_phases=2, grid_n=70)
    wl.phases = np.array([0.5, 0.45])
    one = workloads.make_config2(n_pix=3000, n_phases=2, grid_n=70)
    one.phases = wl.phases
    one.mu_centres = np.array([0.7])
    one.quiet, one.spot = one.quiet[:1].copy(), one.spot[:1].copy()
    assert_parity(one, run_gpu(soap, one))
    many = workloads.make_config2(n_pix=3000, n_phases=2, grid_n=70)
    many.phases = wl.phases
    many.mu_centres = (np.arange(64) + 1.0) / 64.0
    reps = [k * 20 // 64 for k in range(64)]
    many.quiet, many.spot = many.quiet[reps].copy(), many.spot[reps].copy()
    assert_parity(many, run_gpu(soap, many))


def test_pole_on_star_and_polar_and_huge_regions(soap):
    wl = workloads.make_config3(n_pix=3000, n_phases=4, grid_n=64)
    wl.incl_deg = 0.0                                   # pole-on: no Doppler shift at all
    wl.regions = [(90.0, 0.0, 0.3, 2), (10.0, 40.0, 0.95, 1), (-80.0, 200.0, 0.2, 2)]
    wl.phases = np.array([0.0, 0.3, 0.5, 0.9])
    g = run_gpu(soap, wl)
    assert g["n_active"].max() > 500
    assert_parity(wl, g, check_rv=False)
    wl.incl_deg = 12.0
    assert_parity(wl, run_gpu(soap, wl), check_rv=False)


def test_thousands_of_phases_keep_their_order(soap):
    """More phases than the active launch's scheduler ranks by work (f32::kOrderCap = 256): taken as given, same results."""
    wl = workloads.make_config2(n_pix=2048, n_phases=4, grid_n=40)
    base = np.array([0.5, 0.47, 0.0, 0.53])
    wl.phases = np.tile(base, 1100)                      # 4400 phases
    g = run_gpu(soap, wl)
    wl4 = workloads.make_config2(n_pix=2048, n_phases=4, grid_n=40)
    wl4.phases = base
    g4 = run_gpu(soap, wl4)
    assert np.array_equal(g["D"].reshape(1100, 4, -1), np.broadcast_to(g4["D"], (1100, 4, 2048)))
    assert_parity(wl4, g4)


def test_fastest_supported_rotator_and_too_fast(soap):
    wl = workloads.make_config2(n_pix=9000, n_phases=2, grid_n=60)
    wl.vsini_kms = 150.0                                 # halo ~ 250 px at 5000 A
    wl.phases = np.array([0.5, 0.4])
    assert_parity(wl, run_gpu(soap, wl), check_rv=False)
    wl.vsini_kms = 25000.0                               # |v| < 0.1 c, but the staged span would not fit in shared memory
    with pytest.raises(soap.SoapError) as e:
        run_gpu(soap, wl)
    assert e.value.code == soap.binding.SOAP_ERR_UNSUPPORTED


def test_phase_counts_around_the_ordering_cap(soap):
    """255 / 256 / 257 phases of unequal work: ranked heaviest first up to f32::kOrderCap, taken as given beyond it -
    the order in which items are computed must not show in the result."""
    base = workloads.make_config2(n_pix=2300, n_phases=8, grid_n=48)
    base.regions = [(20.0, 180.0, 0.25, 1), (-30.0, 40.0, 0.1, 1)]
    base.phases = np.array([0.5, 0.31, 0.77, 0.02, 0.44, 0.9, 0.62, 0.13])
    g8 = run_gpu(soap, base)
    assert_parity(base, g8, check_rv=False)
    for n in (255, 256, 257):
        wl = workloads.make_config2(n_pix=2300, n_phases=8, grid_n=48)
        wl.regions = base.regions
        wl.phases = np.resize(base.phases, n)
        g = run_gpu(soap, wl)
        assert np.array_equal(g["D"], g8["D"][np.arange(n) % 8])
        assert np.array_equal(g["n_active"], g8["n_active"][np.arange(n) % 8])


def test_grid_too_large_for_the_shared_memory_finalisation(soap):
    """N x n_mu binned weights beyond geometry.cuh's kFinSmemMax (160 KB): the last CTA finalises from global memory."""
    wl = workloads.make_config2(n_pix=2100, n_phases=2, grid_n=1100)
    wl.phases = np.array([0.5, 0.46])
    g = run_gpu(soap, wl)
    og = oracle.geometry(wl)
    assert g["info"]["n_visible"] == og["n_visible"]
    assert abs(g["info"]["sum_weights"] - og["sum_w"]) <= 1e-9 * og["sum_w"]
    assert_parity(wl, g, check_rv=False)


def test_step_captured_in_a_cuda_graph_replays_bit_identically(soap):
    """A single star's step whose region centres travel as kernel arguments (<= 192 (phase, region) pairs, no n_active
    output) enqueues four kernels and nothing else: it can be captured in a CUDA graph and replayed."""
    wl = workloads.make_config3(n_pix=9000, n_phases=6, grid_n=80)
    dev = torch.device("cuda:0")
    star = soap.soap_create(0)
    q = soap.to_device_spectra(wl.quiet, wl.lambda0, wl.dlambda, dev)
    s = soap.to_device_spectra(wl.spot, wl.lambda0, wl.dlambda, dev, wl.spot_contrast, wl.spot_lb)
    f = soap.to_device_spectra(wl.facula, wl.lambda0, wl.dlambda, dev, wl.facula_contrast, wl.facula_lb)
    Q = torch.zeros(wl.n_pix, dtype=torch.float32, device=dev)
    D = torch.zeros((len(wl.phases), wl.n_pix), dtype=torch.float32, device=dev)

    def step():
        soap.soap_disk_geometry(star, wl, want_info=False)
        soap.soap_integrate_quiet(star, q, Q)
        soap.soap_active_timeseries(star, q, s, f, wl.regions, wl.phases, D)

    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        step()                                     # warm-up: every scratch buffer reaches its size outside the capture
        side.synchronize()
        Q0, D0 = Q.clone(), D.clone()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            step()
    for _ in range(3):
        Q.zero_()
        D.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(Q, Q0) and torch.equal(D, D0)
    soap.soap_destroy(star)
    g = dict(Q=Q0.cpu().numpy(), D=D0.cpu().numpy(), n_active=oracle.run_workload(wl)[2])
    assert_parity(wl, g, check_rv=False)


def test_effects_in_one_pass_without_regions_and_with_hidden_regions(soap):
    """The three-output launch with an empty region list, and with phases at which every region is on the far side:
    exact zeros in all three outputs (S19), counts of zero."""
    from test_gpu_parity import _run_effects
    wl = workloads.make_config3(n_pix=4500, n_phases=3, grid_n=60)
    wl.phases = np.array([0.0, 0.5, 0.98])
    wl.regions = []
    outs, na = _run_effects(soap, wl)
    assert list(na) == [0, 0, 0]
    for o in outs:
        assert o.shape == (3, 4500) and np.all(o == 0.0)
    wl.regions = [(10.0, 180.0, 0.15, 1), (-5.0, 170.0, 0.2, 2)]
    outs, na = _run_effects(soap, wl)
    assert na[0] == 0 and na[1] > 0
    for o in outs:
        assert np.all(o[0] == 0.0) and np.any(o[1] != 0.0)
