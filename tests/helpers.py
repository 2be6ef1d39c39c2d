"""Acceptance metrics of BASELINE.json `north_star`, made concrete.

Plain numpy post-processing applied identically to the oracle's and the CUDA path's outputs; none
of it is part of either implementation.
"""
from __future__ import annotations

import numpy as np

C_CMS = 299792.458e5  # cm/s

QUIET_TOL = 1e-5   # max |Q_gpu - Q_oracle| <= QUIET_TOL * sum_w           (north_star)
DELTA_TOL = 1e-4   # max |D_gpu - D_oracle| <= DELTA_TOL * max |D_oracle|  (north_star)
RV_TOL_CMS = 1.0   # per-line first-moment RV difference                   (north_star)


def line_rvs(F, sum_w, lambda0, k, centres, sigmas, m_lo=0, edge_px=0):
    """First-moment RV (cm/s) of every generated line in the spectrum F (pixels m_lo .. m_lo+len(F)-1).

    window |lam - lam_l| <= 3 max(sigma_l, 0.03 A);  f = F / sum_w;
    RV_l = c * sum((lam - lam_l)(1 - f)) / sum(1 - f) / lam_l.
    Lines whose window is not fully inside [m_lo + edge_px, m_lo + len(F) - edge_px) get NaN
    (edge_px = the clamped-end margin, reading S8)."""
    F = np.asarray(F, dtype=np.float64)
    n = F.shape[-1]
    centres = np.asarray(centres, dtype=np.float64)
    half = 3.0 * np.maximum(np.asarray(sigmas, dtype=np.float64), 0.03)
    lo = np.ceil((centres - half - lambda0) / k).astype(np.int64) - m_lo
    hi = np.floor((centres + half - lambda0) / k).astype(np.int64) - m_lo  # inclusive
    ok = (lo >= edge_px) & (hi < n - edge_px)
    W = int((hi - lo).max()) + 1 if len(centres) else 1
    idx = lo[:, None] + np.arange(W)[None, :]
    mask = (idx <= hi[:, None]) & ok[:, None]
    idx = np.clip(idx, 0, n - 1)
    lam_rel = (lambda0 + k * (idx + m_lo)) - centres[:, None]
    out_shape = F.shape[:-1] + (len(centres),)
    Ff = F.reshape(-1, n)
    out = np.full((Ff.shape[0], len(centres)), np.nan)
    for r in range(Ff.shape[0]):
        dep = np.where(mask, 1.0 - Ff[r][idx] / sum_w, 0.0)
        den = dep.sum(axis=1)
        num = (lam_rel * dep).sum(axis=1)
        with np.errstate(invalid="ignore", divide="ignore"):
            rv = C_CMS * num / den / centres
        rv[~ok] = np.nan
        out[r] = rv
    return out.reshape(out_shape)


def check_quiet(Q_gpu, Q_orc, sum_w):
    err = float(np.max(np.abs(np.asarray(Q_gpu, dtype=np.float64) - Q_orc)))
    return err / sum_w


def check_delta(D_gpu, D_orc):
    scale = float(np.max(np.abs(D_orc)))
    err = float(np.max(np.abs(np.asarray(D_gpu, dtype=np.float64) - D_orc)))
    return err / scale if scale > 0 else err


def max_rv_diff(F_gpu, F_orc, sum_w, wl, m_lo=0, edge_px=64):
    a = line_rvs(F_gpu, sum_w, wl.lambda0, wl.dlambda, wl.line_centres, wl.line_sigmas, m_lo, edge_px)
    b = line_rvs(F_orc, sum_w, wl.lambda0, wl.dlambda, wl.line_centres, wl.line_sigmas, m_lo, edge_px)
    d = np.abs(a - b)
    if np.all(np.isnan(d)):
        return 0.0, 0
    return float(np.nanmax(d)), int(np.sum(~np.isnan(d)))
