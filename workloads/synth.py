"""Seeded synthetic workloads C1..C5 (BASELINE.json `configs`, made concrete in DESIGN.md).

Only *inputs* are produced here: spectra on a uniform wavelength grid (PAPER.md:160-162,
Eq. 5), per-mu-bin line shifts standing in for the paper's mu-dependent bisectors
(PAPER.md:332-334), Planck-ratio contrast arrays standing in for the `SOAPcontrast`
output, active-region lists and phases.  None of
the method's own arithmetic (Doppler shift, interpolation, limb darkening, disk geometry,
region membership) lives in this module.

Every config draws from one ``numpy.random.default_rng(SEED_BASE + index)`` in the fixed
order written in each ``make_config*`` function.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

SEED_BASE = 230104259
C_KMS = 299792.458

CONFIG_NAMES = {
    1: "C1 tiny (N=50, 2000 px, fp64)",
    2: "C2 solar-like line window (N=300, 10 000 px, 100 phases)",
    3: "C3 full visible range (N=300, 310 000 px, 25 phases)",
    4: "C4 cool K dwarf, many regions (N=400, 200 000 px, 200 phases)",
    5: "C5 parameter sweep batch (64 stars, N=300, 200 000 px, 50 phases)",
}

SPOT, FACULA = 1, 2


@dataclass
class Workload:
    """One star's worth of inputs, in the vocabulary of the C-ABI (include/soap_b200.h)."""

    name: str
    # star / disk
    grid_n: int
    vsini_kms: float
    incl_deg: float
    ld_u1: float
    ld_u2: float
    mu_centres: np.ndarray  # [n_mu] float64 ascending
    # wavelength grid, Eq. 5
    lambda0: float
    dlambda: float
    n_pix: int
    dtype: np.dtype
    # spectra [n_mu, n_pix]
    quiet: np.ndarray
    spot: Optional[np.ndarray] = None
    facula: Optional[np.ndarray] = None
    # post-shift per-pixel contrast (I_ratio of Eq. 3) or None (== 1)
    spot_contrast: Optional[np.ndarray] = None
    facula_contrast: Optional[np.ndarray] = None
    # limb-brightening polynomial LB(mu) = c0 + c1 mu + c2 mu^2
    # differential rotation omega_1 / omega_0 (-0.18 for the Sun); 0 = solid body
    diff_rot: float = 0.0
    spot_lb: Tuple[float, float, float] = (1.0, 0.0, 0.0)
    facula_lb: Tuple[float, float, float] = (1.0, 0.0, 0.0)
    # active regions, list order matters: (lat_deg, lon_deg, radius, type)
    regions: List[Tuple[float, float, float, int]] = field(default_factory=list)
    phases: np.ndarray = field(default_factory=lambda: np.zeros(0))
    doppler_mode: int = 0
    # generator truth, used only by the RV acceptance metric
    line_centres: np.ndarray = field(default_factory=lambda: np.zeros(0))
    line_sigmas: np.ndarray = field(default_factory=lambda: np.zeros(0))
    line_depths: np.ndarray = field(default_factory=lambda: np.zeros(0))

    @property
    def n_mu(self) -> int:
        return int(self.mu_centres.shape[0])

    @property
    def wavelengths(self) -> np.ndarray:
        return self.lambda0 + self.dlambda * np.arange(self.n_pix, dtype=np.float64)


# --------------------------------------------------------------------------------------
# building blocks
# --------------------------------------------------------------------------------------
def _apply_lines(S: np.ndarray, lambda0: float, k: float, centres: np.ndarray,
                 depths: np.ndarray, sigmas: np.ndarray, row_velocity_kms: np.ndarray) -> None:
    """S[b, :] *= prod_l (1 - depth_l * exp(-(lam - c_lb)^2 / (2 sigma_l^2))), in place.

    c_lb = centre_l * (1 + row_velocity_kms[b] / c): the per-mu line-centre shift that stands
    in for the mu-dependent bisectors.  Profiles are truncated at +-8 sigma (exp(-32) ~ 1e-14).
    """
    n_rows, n_pix = S.shape
    shift = 1.0 + np.asarray(row_velocity_kms, dtype=np.float64) / C_KMS  # [n_rows]
    smin, smax = float(shift.min()), float(shift.max())
    for c, d, s in zip(centres, depths, sigmas):
        lo = int(np.floor((c * smin - 8.0 * s - lambda0) / k))
        hi = int(np.ceil((c * smax + 8.0 * s - lambda0) / k)) + 1
        lo = max(lo, 0)
        hi = min(hi, n_pix)
        if hi <= lo:
            continue
        lam = lambda0 + k * np.arange(lo, hi, dtype=np.float64)
        z = (lam[None, :] - (c * shift)[:, None]) / s
        S[:, lo:hi] *= 1.0 - d * np.exp(-0.5 * z * z)


def planck_ratio(lam_angstrom: np.ndarray, t_active: float, t_quiet: float) -> np.ndarray:
    """B_lambda(t_active) / B_lambda(t_quiet): the quantity `SOAPcontrast` evaluates per pixel
    (PAPER.md:312).  Input preparation, not part of the timed path."""
    hc_over_k = 1.438776877e8  # Angstrom * Kelvin
    xq = hc_over_k / (lam_angstrom * t_quiet)
    xa = hc_over_k / (lam_angstrom * t_active)
    return np.expm1(xq) / np.expm1(xa)


def _cb_velocity_kms(mu_centres: np.ndarray) -> np.ndarray:
    """Convective blueshift of the line centres, linear in mu: -350 m/s at mu = 1, 0 at mu = 0.05
    (BASELINE.json configs[1])."""
    return -0.350 * (mu_centres - 0.05) / 0.95


def _mu20() -> np.ndarray:
    return 0.05 * (np.arange(20, dtype=np.float64) + 1.0)


def _log_uniform(rng, lo, hi, n):
    return np.exp(rng.uniform(np.log(lo), np.log(hi), n))


def _blue_dense_centres(rng, lam_lo, lam_hi, n):
    """Line centres with density proportional to 1 + 2 (lam_hi - lam)/(lam_hi - lam_lo)  (3:1 blue:red)."""
    u = rng.uniform(0.0, 1.0, n)
    # pdf(t) = (1 + 2 (1 - t)) / 2 on t in [0,1]  ->  cdf(t) = (3 t - t^2) / 2 ; invert
    t = (3.0 - np.sqrt(9.0 - 8.0 * u)) / 2.0
    return lam_lo + t * (lam_hi - lam_lo)


def _cast(a: Optional[np.ndarray], dtype) -> Optional[np.ndarray]:
    return None if a is None else np.ascontiguousarray(a.astype(dtype))


# --------------------------------------------------------------------------------------
# C1
# --------------------------------------------------------------------------------------
def make_config1(phases: Optional[np.ndarray] = None) -> Workload:
    """C1: N=50, 2000 px, one mu bin, fp64, one spot (contrast baked into the spot spectrum).

    Draw order: 3 line depths U(0.2,0.8), then 3 centres U(5001,5019).
    Phases default to (p + 1/2)/4: with {0, 1/4, 1/2, 3/4} only phase 1/2 shows the spot
    (reading R-C1).
    """
    rng = np.random.default_rng(SEED_BASE + 1)
    lambda0, k, n_pix = 5000.0, 0.01, 2000
    depths = rng.uniform(0.2, 0.8, 3)
    centres = rng.uniform(5001.0, 5019.0, 3)
    sigmas = np.full(3, 0.05)
    lam = lambda0 + k * np.arange(n_pix, dtype=np.float64)
    prof = np.exp(-0.5 * ((lam[None, :] - centres[:, None]) / sigmas[:, None]) ** 2)
    quiet = 1.0 - (depths[:, None] * prof).sum(axis=0)
    spot = 0.6 * (1.0 - (1.1 * depths[:, None] * prof).sum(axis=0))
    if phases is None:
        phases = (np.arange(4, dtype=np.float64) + 0.5) / 4.0
    return Workload(
        name="C1", grid_n=50, vsini_kms=2.0, incl_deg=90.0, ld_u1=0.29, ld_u2=0.34,
        mu_centres=np.array([1.0]), lambda0=lambda0, dlambda=k, n_pix=n_pix,
        dtype=np.dtype(np.float64), quiet=quiet[None, :].copy(), spot=spot[None, :].copy(),
        regions=[(30.0, 180.0, 0.1, SPOT)], phases=np.asarray(phases, dtype=np.float64),
        line_centres=centres, line_sigmas=sigmas, line_depths=depths,
    )


# --------------------------------------------------------------------------------------
# C2 / C3 / C4 / C5 share one spectrum recipe
# --------------------------------------------------------------------------------------
def _spectra_set(rng, lambda0, k, n_pix, n_lines, mu_centres, blue_dense, with_facula,
                 n_band_heads=0, dtype=np.float32):
    """Quiet / spot / (facula) rows.  Draw order: centres, depths, sigmas, then (if any)
    band-head positions and per-comb-line depths."""
    lam_lo = lambda0
    lam_hi = lambda0 + k * (n_pix - 1)
    if blue_dense:
        centres = _blue_dense_centres(rng, lam_lo + 1.0, lam_hi - 1.0, n_lines)
    else:
        centres = rng.uniform(lam_lo + 1.0, lam_hi - 1.0, n_lines)
    depths = rng.uniform(0.05, 0.9, n_lines)
    sigmas = _log_uniform(rng, 0.02, 0.08, n_lines)
    n_mu = mu_centres.shape[0]
    v_cb = _cb_velocity_kms(mu_centres)
    zero_v = np.zeros(n_mu)

    quiet = np.ones((n_mu, n_pix), dtype=np.float64)
    _apply_lines(quiet, lambda0, k, centres, depths, sigmas, v_cb)
    spot = np.ones((n_mu, n_pix), dtype=np.float64)
    _apply_lines(spot, lambda0, k, centres, np.minimum(1.1 * depths, 0.99), sigmas, zero_v)
    if n_band_heads:
        heads = rng.uniform(lam_lo + 1.0, lam_hi - 30.0, n_band_heads)
        comb_depths = rng.uniform(0.01, 0.1, (n_band_heads, 500))
        comb_c = (heads[:, None] + 0.05 * np.arange(500)[None, :]).ravel()
        keep = comb_c < lam_hi - 1.0
        _apply_lines(spot, lambda0, k, comb_c[keep], comb_depths.ravel()[keep],
                     np.full(int(keep.sum()), 0.03), zero_v)
    facula = None
    if with_facula:
        facula = np.ones((n_mu, n_pix), dtype=np.float64)
        _apply_lines(facula, lambda0, k, centres, 0.95 * depths, sigmas, zero_v)
    return (_cast(quiet, dtype), _cast(spot, dtype), _cast(facula, dtype), centres, depths, sigmas)


def make_config2(n_pix: int = 10_000, n_lines: Optional[int] = None, n_phases: int = 100,
                 grid_n: int = 300) -> Workload:
    """C2: N=300, 5000-5100 A at 0.01 A, 20 mu bins, 400 lines, 1 % spot at lat 20, 100 phases, fp32."""
    rng = np.random.default_rng(SEED_BASE + 2)
    lambda0, k = 5000.0, 0.01
    if n_lines is None:
        n_lines = max(4, int(round(400 * n_pix / 10_000)))
    mu = _mu20()
    quiet, spot, _, c, d, s = _spectra_set(rng, lambda0, k, n_pix, n_lines, mu, False, False)
    lam = lambda0 + k * np.arange(n_pix, dtype=np.float64)
    return Workload(
        name="C2", grid_n=grid_n, vsini_kms=2.0, incl_deg=90.0, ld_u1=0.29, ld_u2=0.34,
        mu_centres=mu, lambda0=lambda0, dlambda=k, n_pix=n_pix, dtype=np.dtype(np.float32),
        quiet=quiet, spot=spot,
        spot_contrast=planck_ratio(lam, 4700.0, 5778.0).astype(np.float32),
        regions=[(20.0, 180.0, 0.1, SPOT)],
        phases=np.arange(n_phases, dtype=np.float64) / n_phases,
        line_centres=c, line_sigmas=s, line_depths=d,
    )


def make_config3(n_pix: int = 310_000, n_lines: Optional[int] = None, n_phases: int = 25,
                 grid_n: int = 300, nested: bool = False) -> Workload:
    """C3 (the benchmark workload): N=300, 3800-6900 A at 0.01 A, 20 mu bins x {quiet, spot, facula},
    25 000 lines (3:1 blue:red), 3 % facula then 1 % spot, 25 phases, fp32.

    ``nested=True`` gives the spot-inside-facula variant of PAPER.md:284 (both at lat 30, lon 180)."""
    rng = np.random.default_rng(SEED_BASE + 3)
    lambda0, k = 3800.0, 0.01
    if n_lines is None:
        n_lines = max(8, int(round(25_000 * n_pix / 310_000)))
    mu = _mu20()
    quiet, spot, facula, c, d, s = _spectra_set(rng, lambda0, k, n_pix, n_lines, mu, True, True)
    lam = lambda0 + k * np.arange(n_pix, dtype=np.float64)
    if nested:
        regions = [(30.0, 180.0, float(np.sqrt(0.03)), FACULA), (30.0, 180.0, 0.1, SPOT)]
    else:
        regions = [(-25.0, 60.0, float(np.sqrt(0.03)), FACULA), (20.0, 180.0, 0.1, SPOT)]
    return Workload(
        name="C3", grid_n=grid_n, vsini_kms=2.0, incl_deg=90.0, ld_u1=0.29, ld_u2=0.34,
        mu_centres=mu, lambda0=lambda0, dlambda=k, n_pix=n_pix, dtype=np.dtype(np.float32),
        quiet=quiet, spot=spot, facula=facula,
        spot_contrast=planck_ratio(lam, 4700.0, 5778.0).astype(np.float32),
        facula_contrast=None, facula_lb=(1.1, -0.1, 0.0),
        regions=regions, phases=np.arange(n_phases, dtype=np.float64) / n_phases,
        line_centres=c, line_sigmas=s, line_depths=d,
    )


def make_config4(n_pix: int = 200_000, n_lines: Optional[int] = None, n_phases: int = 200,
                 grid_n: int = 400, n_band_heads: Optional[int] = None) -> Workload:
    """C4: N=400, vsini=3, i=60, LD (0.55,0.15), 4500-6500 A, spot rows with molecular-band combs,
    10 seeded regions, 200 phases, fp32.  Region draw order (after the spectra): type, lat, lon, radius."""
    rng = np.random.default_rng(SEED_BASE + 4)
    lambda0, k = 4500.0, 0.01
    if n_lines is None:
        n_lines = max(8, int(round(16_000 * n_pix / 200_000)))
    if n_band_heads is None:
        n_band_heads = max(1, int(round(40 * n_pix / 200_000)))
    mu = _mu20()
    quiet, spot, facula, c, d, s = _spectra_set(rng, lambda0, k, n_pix, n_lines, mu, True, True,
                                                n_band_heads=n_band_heads)
    lam = lambda0 + k * np.arange(n_pix, dtype=np.float64)
    types = np.where(rng.uniform(0, 1, 10) < 0.5, SPOT, FACULA)
    lats = rng.uniform(-60.0, 60.0, 10)
    lons = rng.uniform(0.0, 360.0, 10)
    radii = rng.uniform(0.02, 0.1, 10)
    regions = [(float(a), float(b), float(r), int(t)) for a, b, r, t in zip(lats, lons, radii, types)]
    return Workload(
        name="C4", grid_n=grid_n, vsini_kms=3.0, incl_deg=60.0, ld_u1=0.55, ld_u2=0.15,
        mu_centres=mu, lambda0=lambda0, dlambda=k, n_pix=n_pix, dtype=np.dtype(np.float32),
        quiet=quiet, spot=spot, facula=facula,
        spot_contrast=planck_ratio(lam, 3500.0, 4500.0).astype(np.float32),
        facula_contrast=None, facula_lb=(1.1, -0.1, 0.0),
        regions=regions, phases=np.arange(n_phases, dtype=np.float64) / n_phases,
        line_centres=c, line_sigmas=s, line_depths=d,
    )


def make_config5_star(star: int, n_pix: int = 200_000, n_lines: Optional[int] = None,
                      n_phases: int = 50, grid_n: int = 300, shared=None) -> Workload:
    """Star `star` (0..63) of the C5 parameter sweep.  The spectra set is shared by all stars
    (drawn first from the config rng); each star then has its own child rng
    ``default_rng([SEED_BASE + 5, star])`` with draw order vsini, incl, u1, u2, n_regions,
    then per region type, lat, lon, radius.  Pass ``shared`` (a previous Workload of this config
    with the same n_pix) to reuse the spectra arrays instead of regenerating them."""
    lambda0, k = 4500.0, 0.01
    mu = _mu20()
    if shared is None:
        rng = np.random.default_rng(SEED_BASE + 5)
        if n_lines is None:
            n_lines = max(8, int(round(8_000 * n_pix / 200_000)))
        quiet, spot, facula, c, d, s = _spectra_set(rng, lambda0, k, n_pix, n_lines, mu, False, True)
        lam = lambda0 + k * np.arange(n_pix, dtype=np.float64)
        contrast = planck_ratio(lam, 4700.0, 5778.0).astype(np.float32)
    else:
        quiet, spot, facula = shared.quiet, shared.spot, shared.facula
        c, d, s = shared.line_centres, shared.line_depths, shared.line_sigmas
        contrast = shared.spot_contrast
    srng = np.random.default_rng([SEED_BASE + 5, int(star)])
    vsini = float(_log_uniform(srng, 1.0, 20.0, 1)[0])
    incl = float(srng.uniform(20.0, 90.0))
    u1 = float(srng.uniform(0.2, 0.6))
    u2 = float(srng.uniform(0.2, 0.6))
    n_reg = int(srng.integers(1, 6))
    regions = []
    for _ in range(n_reg):
        t = SPOT if srng.uniform() < 0.5 else FACULA
        lat = float(srng.uniform(-60.0, 60.0))
        lon = float(srng.uniform(0.0, 360.0))
        rad = float(srng.uniform(0.02, 0.1))
        regions.append((lat, lon, rad, t))
    return Workload(
        name=f"C5[{star}]", grid_n=grid_n, vsini_kms=vsini, incl_deg=incl, ld_u1=u1, ld_u2=u2,
        mu_centres=mu, lambda0=lambda0, dlambda=k, n_pix=n_pix, dtype=np.dtype(np.float32),
        quiet=quiet, spot=spot, facula=facula, spot_contrast=contrast,
        facula_contrast=None, facula_lb=(1.1, -0.1, 0.0),
        regions=regions, phases=np.arange(n_phases, dtype=np.float64) / n_phases,
        line_centres=c, line_sigmas=s, line_depths=d,
    )


def make_workload(config: int, **kw) -> Workload:
    if config == 1:
        return make_config1(**kw)
    if config == 2:
        return make_config2(**kw)
    if config == 3:
        return make_config3(**kw)
    if config == 4:
        return make_config4(**kw)
    if config == 5:
        return make_config5_star(kw.pop("star", 0), **kw)
    raise ValueError(f"unknown config {config}")


# ---- active-region size evolution: input preparation for soap_active_timeseries_evolving ----
MSH = 1e-6  # one millionth of the solar hemisphere; reading S11: filling factor f <-> radius sqrt(f)


def evolution_radii(kind: str, t_days: np.ndarray, size0_msh: float = 10_000.0, rate_msh_per_day: float = 400.0,
                    fwhm_days: float = 10.0, asymmetry: float = 0.09, t_peak_days: float = 0.0) -> np.ndarray:
    """Radius (stellar radii) of one region at the times t_days under the three laws of P:280:
    'growth' / 'decay': size(t) = size0 +/- rate t;  'gaussian': size0 exp(-(t - t_peak)^2 / 2 sigma^2) with
    sigma = FWHM / 2.3548 * (1 -/+ asymmetry) before / after the peak (a stand-in for Murakozy et al. 2014, whose
    exact form the paper does not give).  Sizes in MSH, clipped at 0; radius = sqrt(size * 1e-6)."""
    t = np.asarray(t_days, dtype=np.float64)
    if kind == "growth":
        size = size0_msh + rate_msh_per_day * t
    elif kind == "decay":
        size = size0_msh - rate_msh_per_day * t
    elif kind == "gaussian":
        s0 = fwhm_days / (2.0 * np.sqrt(2.0 * np.log(2.0)))
        sig = np.where(t < t_peak_days, s0 * (1.0 - asymmetry), s0 * (1.0 + asymmetry))
        size = size0_msh * np.exp(-((t - t_peak_days) ** 2) / (2.0 * sig * sig))
    else:
        raise ValueError("kind must be 'growth', 'decay' or 'gaussian'")
    return np.sqrt(np.clip(size, 0.0, None) * MSH)
