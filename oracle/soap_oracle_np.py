"""TEST INFRASTRUCTURE - numpy twin of oracle/soap_oracle.c for tiny sizes.

The same definition (Alg. 1, Eq. 3, InfoMap P:208 of /root/reference/PAPER.md),
written with ``numpy.interp`` as the per-cell shift+interpolate step (Alg. 1 lines 3-4; its
clamp-to-edge rule is reading S8 of DESIGN.md).  Pure-Python loops over cells: use only for
small grids.  Shares nothing with the CUDA path and does not import the C oracle either - the
two are compared against each other in tests/test_oracle_pins.py (pin P8).
"""
from __future__ import annotations

import math

import numpy as np

C_KMS = 299792.458


def doppler_factor(v_kms: float, mode: int) -> float:
    beta = v_kms / C_KMS
    if mode == 1:
        return 1.0 - beta
    return math.sqrt((1.0 - beta) / (1.0 + beta))  # Eq. 6, inverted (gather)


def geometry(grid_n, vsini_kms, incl_deg, u1, u2, mu_centres, doppler_mode=0, diff_rot=0.0):
    """List of visible cells as dicts, in (j, i) order (readings S1-S5, S9).  diff_rot = omega_1 / omega_0 of
    omega = omega_0 + omega_1 sin^2(latitude) (reading R-DR)."""
    N = grid_n
    mu_centres = np.asarray(mu_centres, dtype=np.float64)
    sini = math.sin(math.radians(incl_deg))
    cosi = math.cos(math.radians(incl_deg))
    cells = []
    for j in range(N):
        for i in range(N):
            x = -1.0 + (2.0 * j + 1.0) / N
            y = -1.0 + (2.0 * i + 1.0) / N
            r2 = x * x + y * y
            if r2 > 1.0:
                continue
            mu = math.sqrt(max(0.0, 1.0 - r2))
            v = x * vsini_kms * sini
            if diff_rot != 0.0:
                v *= 1.0 + diff_rot * (y * sini + mu * cosi) ** 2  # sin(latitude) of the surface point (x, y, mu)
            w = 1.0 - u1 * (1.0 - mu) - u2 * (1.0 - mu) ** 2
            d = np.abs(mu - mu_centres)
            b = int(np.flatnonzero(d == d.min())[-1])  # tie -> larger mu
            cells.append(dict(j=j, i=i, x=x, y=y, mu=mu, v=v, w=w, bin=b,
                              D=doppler_factor(v, doppler_mode)))
    return cells


def quiet(cells, S, lambda0, k):
    """Alg. 1: Q = sum_cells w * interp(lam * D, lam, S[bin])."""
    S = np.asarray(S, dtype=np.float64)
    P = S.shape[1]
    lam = lambda0 + k * np.arange(P, dtype=np.float64)
    Q = np.zeros(P)
    for c in cells:
        Q += c["w"] * np.interp(lam * c["D"], lam, S[c["bin"]])
    return Q


def region_centre(lat_deg, lon_deg, incl_deg, phase):
    lat = math.radians(lat_deg)
    L = math.radians(lon_deg) + 2.0 * math.pi * phase
    inc = math.radians(incl_deg)
    sx, sy, sz = math.cos(lat) * math.sin(L), math.sin(lat), math.cos(lat) * math.cos(L)
    return sx, sy * math.sin(inc) - sz * math.cos(inc), sy * math.cos(inc) + sz * math.sin(inc)


def info_map(cells, regions, incl_deg, phase):
    """type per visible cell: last covering region in list order wins."""
    types = [0] * len(cells)
    for (lat, lon, radius, rtype) in regions:
        xr, yr, zr = region_centre(lat, lon, incl_deg, phase)
        cos_alpha = math.sqrt(1.0 - radius * radius)
        for n, c in enumerate(cells):
            if c["x"] * xr + c["y"] * yr + c["mu"] * zr >= cos_alpha:
                types[n] = rtype
    return types


def active(cells, incl_deg, S_quiet, S_spot, S_facula, C_spot, C_facula, lb_spot, lb_facula,
           lambda0, k, regions, phases, effect=0):
    """delta[p] = sum_active w (C_t LB_t(mu) shifted(S_t[bin]) - shifted(S_quiet[bin]))  (Eq. 3, north_star sign).
    effect 1: flux only, w (I_ratio shifted(S_quiet) - shifted(S_quiet)) (Eq. 1); effect 2: convective blueshift
    only, w (shifted(S_t) - shifted(S_quiet)) (Eq. 2)."""
    S_quiet = np.asarray(S_quiet, dtype=np.float64)
    P = S_quiet.shape[1]
    lam = lambda0 + k * np.arange(P, dtype=np.float64)
    out = np.zeros((len(phases), P))
    n_active = []
    for p, ph in enumerate(phases):
        types = info_map(cells, regions, incl_deg, ph)
        n_active.append(sum(1 for t in types if t))
        for c, t in zip(cells, types):
            if t == 0:
                continue
            Sa = np.asarray(S_spot if t == 1 else S_facula, dtype=np.float64)
            C = C_spot if t == 1 else C_facula
            lbc = lb_spot if t == 1 else lb_facula
            lb = lbc[0] + lbc[1] * c["mu"] + lbc[2] * c["mu"] ** 2
            cm = 1.0 if C is None else np.asarray(C, dtype=np.float64)
            x = lam * c["D"]
            sq = np.interp(x, lam, S_quiet[c["bin"]])
            sa = np.interp(x, lam, Sa[c["bin"]])
            if effect == 0:
                out[p] += c["w"] * (cm * lb * sa - sq)
            elif effect == 1:
                out[p] += c["w"] * (cm * lb * sq - sq)
            elif effect == 2:
                out[p] += c["w"] * (sa - sq)
            else:
                raise ValueError("effect must be 0, 1 or 2")
    return out, n_active
