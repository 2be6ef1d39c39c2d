"""TEST INFRASTRUCTURE - ctypes front end of the fp64 CPU oracle (oracle/soap_oracle.c).

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It never imports the CUDA path (paper_2301_04259_b200) and the
CUDA path never imports it.

Star-like arguments are duck-typed: any object with attributes grid_n, vsini_kms, incl_deg,
ld_u1, ld_u2, mu_centres, doppler_mode (workloads.Workload has them).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "soap_oracle.c")
_LIB = os.path.join(_HERE, "libsoap_oracle.so")
_lib = None


class _Star(ctypes.Structure):
    _fields_ = [("grid_n", ctypes.c_int32), ("vsini_kms", ctypes.c_double), ("incl_deg", ctypes.c_double),
                ("ld_u1", ctypes.c_double), ("ld_u2", ctypes.c_double), ("n_mu", ctypes.c_int32),
                ("mu_centres", ctypes.POINTER(ctypes.c_double)), ("doppler_mode", ctypes.c_int32),
                ("diff_rot", ctypes.c_double)]


class _Region(ctypes.Structure):
    _fields_ = [("lat_deg", ctypes.c_double), ("lon_deg", ctypes.c_double), ("radius", ctypes.c_double),
                ("type", ctypes.c_int32)]


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc -O2 -fopenmp (no -ffast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.soap_oracle_num_threads.restype = ctypes.c_int
        lib.soap_oracle_set_threads.argtypes = [ctypes.c_int]
        lib.soap_oracle_geometry.restype = ctypes.c_int64
        lib.soap_oracle_geometry.argtypes = [ctypes.POINTER(_Star)] + [ctypes.c_void_p] * 9
        lib.soap_oracle_shifted_row.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_double,
                                                ctypes.c_double, ctypes.c_double, ctypes.c_int64,
                                                ctypes.c_int64, ctypes.c_void_p]
        lib.soap_oracle_quiet.restype = ctypes.c_int
        lib.soap_oracle_quiet.argtypes = [ctypes.POINTER(_Star), ctypes.c_void_p, ctypes.c_int64,
                                          ctypes.c_double, ctypes.c_double, ctypes.c_int64, ctypes.c_int64,
                                          ctypes.c_void_p]
        lib.soap_oracle_info_map.restype = ctypes.c_int64
        lib.soap_oracle_info_map.argtypes = [ctypes.POINTER(_Star), ctypes.POINTER(_Region), ctypes.c_int32,
                                             ctypes.c_double, ctypes.c_void_p]
        lib.soap_oracle_active.restype = ctypes.c_int
        lib.soap_oracle_active.argtypes = [ctypes.POINTER(_Star)] + [ctypes.c_void_p] * 7 + [
            ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.POINTER(_Region), ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        lib.soap_oracle_active_effect.restype = ctypes.c_int
        lib.soap_oracle_active_effect.argtypes = [ctypes.POINTER(_Star)] + [ctypes.c_void_p] * 7 + [
            ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.POINTER(_Region), ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p,
            ctypes.c_void_p]
        lib.soap_oracle_lower_resolution.restype = ctypes.c_int
        lib.soap_oracle_lower_resolution.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_double,
                                                     ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_void_p]
        lib.soap_oracle_line_rvs.restype = ctypes.c_int
        lib.soap_oracle_line_rvs.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_double, ctypes.c_double,
                                             ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64,
                                             ctypes.c_void_p]
        lib.soap_oracle_contrast_planck.restype = ctypes.c_int
        lib.soap_oracle_contrast_planck.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int64, ctypes.c_double,
                                                    ctypes.c_double, ctypes.c_void_p]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().soap_oracle_num_threads())


def set_threads(n: int) -> None:
    _load().soap_oracle_set_threads(int(n))


def _star(s):
    mu = np.ascontiguousarray(np.asarray(s.mu_centres, dtype=np.float64))
    st = _Star(int(s.grid_n), float(s.vsini_kms), float(s.incl_deg), float(s.ld_u1), float(s.ld_u2),
               int(mu.shape[0]), mu.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
               int(getattr(s, "doppler_mode", 0)), float(getattr(s, "diff_rot", 0.0)))
    return st, mu  # keep mu alive


def _f64(a) -> Optional[np.ndarray]:
    return None if a is None else np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data


def _regions(regions: Sequence):
    arr = (_Region * max(1, len(regions)))()
    for n, (lat, lon, rad, typ) in enumerate(regions):
        arr[n] = _Region(float(lat), float(lon), float(rad), int(typ))
    return arr


def geometry(star) -> dict:
    """Per-cell arrays (N*N, index j*N+i): x, y, mu, vel, w, D, bin, visible; plus n_visible, sum_w."""
    lib = _load()
    st, _keep = _star(star)
    n = int(star.grid_n) ** 2
    out = {k: np.zeros(n, dtype=np.float64) for k in ("x", "y", "mu", "vel", "w", "D")}
    out["bin"] = np.zeros(n, dtype=np.int32)
    out["visible"] = np.zeros(n, dtype=np.uint8)
    sw = ctypes.c_double(0.0)
    nv = lib.soap_oracle_geometry(ctypes.byref(st), out["x"].ctypes.data, out["y"].ctypes.data,
                                  out["mu"].ctypes.data, out["vel"].ctypes.data, out["w"].ctypes.data,
                                  out["D"].ctypes.data, out["bin"].ctypes.data, out["visible"].ctypes.data,
                                  ctypes.addressof(sw))
    out["n_visible"] = int(nv)
    out["sum_w"] = float(sw.value)
    return out


def shifted_row(S, lambda0: float, k: float, D: float, m_lo: int = 0, m_hi: Optional[int] = None):
    lib = _load()
    S = _f64(S)
    P = S.shape[0]
    m_hi = P if m_hi is None else m_hi
    out = np.zeros(m_hi - m_lo, dtype=np.float64)
    lib.soap_oracle_shifted_row(S.ctypes.data, P, float(lambda0), float(k), float(D), int(m_lo), int(m_hi),
                                out.ctypes.data)
    return out


def quiet(star, S_quiet, lambda0: float, k: float, m_lo: int = 0, m_hi: Optional[int] = None) -> np.ndarray:
    """Alg. 1 over pixels [m_lo, m_hi).  S_quiet: [n_mu, P] (any float dtype; promoted exactly to fp64)."""
    lib = _load()
    st, _keep = _star(star)
    S = _f64(S_quiet)
    assert S.ndim == 2 and S.shape[0] == st.n_mu
    P = S.shape[1]
    m_hi = P if m_hi is None else m_hi
    out = np.zeros(m_hi - m_lo, dtype=np.float64)
    rc = lib.soap_oracle_quiet(ctypes.byref(st), S.ctypes.data, P, float(lambda0), float(k), int(m_lo),
                               int(m_hi), out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"soap_oracle_quiet failed: {rc}")
    return out


def info_map(star, regions: Sequence, phase: float):
    lib = _load()
    st, _keep = _star(star)
    tm = np.zeros(int(star.grid_n) ** 2, dtype=np.int32)
    n = lib.soap_oracle_info_map(ctypes.byref(st), _regions(regions), len(regions), float(phase), tm.ctypes.data)
    return tm, int(n)


def active(star, S_quiet, S_spot, S_facula, lambda0: float, k: float, regions: Sequence, phases,
           C_spot=None, C_facula=None, lb_spot=(1.0, 0.0, 0.0), lb_facula=(1.0, 0.0, 0.0),
           m_lo: int = 0, m_hi: Optional[int] = None, effect: int = 0):
    """Alg. 5 + Eq. 3 (north_star sign) over pixels [m_lo, m_hi).  Returns (delta [n_ph, n], n_active [n_ph]).
    effect: 0 = total (Eq. 3), 1 = flux only (Eq. 1), 2 = convective blueshift only (Eq. 2)."""
    lib = _load()
    st, _keep = _star(star)
    Sq, Ss, Sf = _f64(S_quiet), _f64(S_spot), _f64(S_facula)
    Cs, Cf = _f64(C_spot), _f64(C_facula)
    lbs, lbf = _f64(lb_spot), _f64(lb_facula)
    P = Sq.shape[1]
    m_hi = P if m_hi is None else m_hi
    ph = _f64(phases)
    delta = np.zeros((ph.shape[0], m_hi - m_lo), dtype=np.float64)
    n_active = np.zeros(ph.shape[0], dtype=np.int32)
    rc = lib.soap_oracle_active_effect(ctypes.byref(st), _ptr(Sq), _ptr(Ss), _ptr(Sf), _ptr(Cs), _ptr(Cf),
                                       _ptr(lbs), _ptr(lbf), P, float(lambda0), float(k), _regions(regions),
                                       len(regions), ph.ctypes.data, ph.shape[0], int(m_lo), int(m_hi),
                                       int(effect), delta.ctypes.data, n_active.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"soap_oracle_active failed: {rc}")
    return delta, n_active


def run_workload(wl, m_lo: int = 0, m_hi: Optional[int] = None, effect: int = 0):
    """Convenience: (Q, delta, n_active, geometry-info) of a workloads.Workload-like object."""
    Q = quiet(wl, wl.quiet, wl.lambda0, wl.dlambda, m_lo, m_hi)
    delta, n_active = active(wl, wl.quiet, wl.spot, wl.facula, wl.lambda0, wl.dlambda, wl.regions,
                             wl.phases, wl.spot_contrast, wl.facula_contrast, wl.spot_lb, wl.facula_lb,
                             m_lo, m_hi, effect)
    return Q, delta, n_active


LSF_NSIG = 5.0  # truncation of the line-spread function in sigmas (reading R-LSF)


def lower_resolution(rows, lambda0: float, k: float, R: float, nsig: float = LSF_NSIG) -> np.ndarray:
    """Resolution lowering of PAPER.md:85 / Alg. 5 P:244 with a Gaussian LSF of FWHM lambda/R (reading R-LSF).
    rows: [n_rows, P] (or [P]); returns the same shape in fp64."""
    lib = _load()
    a = _f64(np.atleast_2d(rows))
    out = np.empty_like(a)
    rc = lib.soap_oracle_lower_resolution(a.ctypes.data, a.shape[0], a.shape[1], float(lambda0), float(k), float(R),
                                          float(nsig), out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"soap_oracle_lower_resolution failed: {rc}")
    return out.reshape(np.shape(rows))


def active_evolving(star, S_quiet, S_spot, S_facula, lambda0: float, k: float, regions: Sequence, phases, radii,
                    C_spot=None, C_facula=None, lb_spot=(1.0, 0.0, 0.0), lb_facula=(1.0, 0.0, 0.0),
                    m_lo: int = 0, m_hi: Optional[int] = None, effect: int = 0):
    """Evolving regions: phase p sees region r with radius radii[p][r] (<= 0: absent).  Plain loop
    over the phases around `active` (Alg. 5 is per timestep: the region list is simply different at every step)."""
    radii = np.asarray(radii, dtype=np.float64).reshape(len(phases), len(regions))
    rows, counts = [], []
    for p, ph in enumerate(phases):
        regs = [(lat, lon, float(radii[p][r]), typ) for r, (lat, lon, _rad, typ) in enumerate(regions) if radii[p][r] > 0.0]
        d, n = active(star, S_quiet, S_spot, S_facula, lambda0, k, regs, np.array([ph], dtype=np.float64), C_spot, C_facula,
                      lb_spot, lb_facula, m_lo, m_hi, effect)
        rows.append(d[0])
        counts.append(int(n[0]))
    return np.stack(rows), np.asarray(counts, dtype=np.int32)


def line_rvs(rows, lambda0: float, k: float, centres, half_widths, norm, edge: int = 0) -> np.ndarray:
    """First-moment RV (cm/s) of every line in every row (north_star's acceptance functional).
    rows [n_rows, P] (or [P]); norm: scalar or [n_rows] continuum level; returns [n_rows, n_lines] (NaN: window off-grid)."""
    lib = _load()
    a = _f64(np.atleast_2d(rows))
    c, h = _f64(np.atleast_1d(centres)), _f64(np.atleast_1d(half_widths))
    nrm = _f64(np.broadcast_to(np.asarray(norm, dtype=np.float64), (a.shape[0],)).copy())
    out = np.empty((a.shape[0], c.shape[0]), dtype=np.float64)
    rc = lib.soap_oracle_line_rvs(a.ctypes.data, a.shape[0], a.shape[1], float(lambda0), float(k), c.ctypes.data, h.ctypes.data,
                                  c.shape[0], nrm.ctypes.data, int(edge), out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"soap_oracle_line_rvs failed: {rc}")
    return out


def contrast_planck(lambda0: float, k: float, n_pix: int, t_quiet: float, t_active: float) -> np.ndarray:
    """SOAPcontrast: B_lambda(t_active) / B_lambda(t_quiet) at lambda_m = lambda0 + m k (Angstrom), fp64."""
    lib = _load()
    out = np.empty(int(n_pix), dtype=np.float64)
    rc = lib.soap_oracle_contrast_planck(float(lambda0), float(k), int(n_pix), float(t_quiet), float(t_active), out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"soap_oracle_contrast_planck failed: {rc}")
    return out
