"""Thin Python binding of the C ABI in include/soap_b200.h (argument marshalling only).

Every function here has the name and the semantics of the C entry point it wraps; all computation
happens in the CUDA kernels behind ``libsoap_b200.so``.  PyTorch is used for device memory
(``tensor.data_ptr()``) and streams (``torch.cuda.current_stream().cuda_stream``) and nothing else.
There is no fallback: if the shared library has not been built, importing this module raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence, Tuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsoap_b200.so")

SOAP_OK = 0
SOAP_ERR_INVALID_ARG, SOAP_ERR_NOT_READY, SOAP_ERR_CUDA, SOAP_ERR_OOM, SOAP_ERR_UNSUPPORTED = -1, -2, -3, -4, -5
SOAP_F32, SOAP_F64 = 0, 1
SOAP_SPOT, SOAP_FACULA = 1, 2
SOAP_FORM_AUTO, SOAP_FORM_BINNED, SOAP_FORM_CELLS, SOAP_FORM_FIR, SOAP_FORM_COMPOSITE = 0, 1, 2, 3, 4
SOAP_OPT_FORM, SOAP_OPT_QUIET_SPLITS, SOAP_OPT_KERNEL_TIMING, SOAP_OPT_EFFECT_PASSES = 1, 2, 3, 4

EXPORTED_SYMBOLS = (
    "soap_version", "soap_create", "soap_destroy", "soap_last_error", "soap_set_option", "soap_get_stats",
    "soap_disk_geometry", "soap_integrate_quiet", "soap_active_timeseries", "soap_active_timeseries_effects",
    "soap_export_geometry", "soap_lower_resolution", "soap_active_timeseries_evolving", "soap_line_rvs",
    "soap_synthesize_host", "soap_batch_integrate_quiet", "soap_batch_active_timeseries", "soap_contrast_planck",
    "soap_batch_disk_geometry", "soap_integrate_quiet_static",
)


class SoapError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"soap error {code}: {message}")
        self.code = code
        self.message = message


class c_star_params(ctypes.Structure):
    _fields_ = [("grid_n", ctypes.c_int32), ("vsini_kms", ctypes.c_double), ("incl_deg", ctypes.c_double),
                ("ld_u1", ctypes.c_double), ("ld_u2", ctypes.c_double), ("n_mu", ctypes.c_int32),
                ("mu_centres", ctypes.POINTER(ctypes.c_double)), ("doppler_mode", ctypes.c_int32),
                ("diff_rot", ctypes.c_double)]


class c_spectra(ctypes.Structure):
    _fields_ = [("data", ctypes.c_void_p), ("n_pix", ctypes.c_int64), ("pitch", ctypes.c_int64),
                ("dtype", ctypes.c_int32), ("lambda0", ctypes.c_double), ("dlambda", ctypes.c_double),
                ("contrast", ctypes.c_void_p), ("lb_c0", ctypes.c_double), ("lb_c1", ctypes.c_double),
                ("lb_c2", ctypes.c_double)]


class c_region(ctypes.Structure):
    _fields_ = [("lat_deg", ctypes.c_double), ("lon_deg", ctypes.c_double), ("radius", ctypes.c_double),
                ("type", ctypes.c_int32)]


class c_geom_info(ctypes.Structure):
    _fields_ = [("n_visible", ctypes.c_int64), ("n_entries", ctypes.c_int64), ("sum_weights", ctypes.c_double),
                ("max_abs_dshift", ctypes.c_double)]


class c_stats(ctypes.Structure):
    _fields_ = [("quiet_entries", ctypes.c_int64), ("active_entries", ctypes.c_int64),
                ("active_cells", ctypes.c_int64), ("quiet_splits", ctypes.c_int32), ("tile_px", ctypes.c_int32),
                ("form", ctypes.c_int32), ("launches", ctypes.c_int32), ("quiet_kernel_ms", ctypes.c_float),
                ("active_kernel_ms", ctypes.c_float)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libsoap_b200.so and declare the prototypes.  Raises ImportError if it was not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2301_04259_b200.build` "
            "(or __graft_entry__.build()).  There is no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    lib.soap_version.restype = ctypes.c_int
    lib.soap_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int]
    lib.soap_destroy.argtypes = [vp]
    lib.soap_last_error.argtypes = [vp]
    lib.soap_last_error.restype = ctypes.c_char_p
    lib.soap_set_option.argtypes = [vp, i32, i64]
    lib.soap_get_stats.argtypes = [vp, ctypes.POINTER(c_stats), vp]
    lib.soap_disk_geometry.argtypes = [vp, ctypes.POINTER(c_star_params), vp, ctypes.POINTER(c_geom_info)]
    lib.soap_integrate_quiet.argtypes = [vp, ctypes.POINTER(c_spectra), vp, vp]
    lib.soap_integrate_quiet_static.argtypes = [vp, ctypes.POINTER(c_spectra), vp, vp]
    lib.soap_active_timeseries.argtypes = [vp, ctypes.POINTER(c_spectra), ctypes.POINTER(c_spectra),
                                           ctypes.POINTER(c_spectra), ctypes.POINTER(c_region), i32,
                                           ctypes.POINTER(ctypes.c_double), i32, vp, i64,
                                           ctypes.POINTER(i32), vp]
    lib.soap_active_timeseries_effects.argtypes = [vp, ctypes.POINTER(c_spectra), ctypes.POINTER(c_spectra),
                                                   ctypes.POINTER(c_spectra), ctypes.POINTER(c_region), i32,
                                                   ctypes.POINTER(ctypes.c_double), i32, vp, vp, vp, i64,
                                                   ctypes.POINTER(i32), vp]
    lib.soap_export_geometry.argtypes = [vp, vp, vp, vp, vp]
    lib.soap_contrast_planck.argtypes = [vp, ctypes.c_double, ctypes.c_double, i64, ctypes.c_double, ctypes.c_double, vp, i32, vp]
    lib.soap_line_rvs.argtypes = [vp, vp, i64, i64, i64, i32, ctypes.c_double, ctypes.c_double, vp, vp, i64, vp, i64, vp, vp]
    lib.soap_active_timeseries_evolving.argtypes = [vp, ctypes.POINTER(c_spectra), ctypes.POINTER(c_spectra),
                                                    ctypes.POINTER(c_spectra), ctypes.POINTER(c_region), i32,
                                                    ctypes.POINTER(ctypes.c_double), i32, ctypes.POINTER(ctypes.c_double),
                                                    vp, vp, vp, i64, ctypes.POINTER(i32), vp]
    lib.soap_lower_resolution.argtypes = [vp, vp, i64, i64, i64, i32, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                          vp, i64, vp]
    lib.soap_synthesize_host.argtypes = [vp, ctypes.POINTER(c_star_params), ctypes.POINTER(c_spectra),
                                         ctypes.POINTER(c_spectra), ctypes.POINTER(c_spectra),
                                         ctypes.POINTER(c_region), i32, ctypes.POINTER(ctypes.c_double), i32,
                                         vp, vp, ctypes.POINTER(i32), vp]
    lib.soap_batch_disk_geometry.argtypes = [ctypes.POINTER(vp), i32, ctypes.POINTER(ctypes.POINTER(c_star_params)), vp,
                                             ctypes.POINTER(c_geom_info)]
    lib.soap_batch_integrate_quiet.argtypes = [ctypes.POINTER(vp), i32, ctypes.POINTER(ctypes.POINTER(c_spectra)),
                                               ctypes.POINTER(vp), vp]
    lib.soap_batch_active_timeseries.argtypes = [
        ctypes.POINTER(vp), i32, ctypes.POINTER(ctypes.POINTER(c_spectra)),
        ctypes.POINTER(ctypes.POINTER(c_spectra)), ctypes.POINTER(ctypes.POINTER(c_spectra)),
        ctypes.POINTER(ctypes.POINTER(c_region)), ctypes.POINTER(i32),
        ctypes.POINTER(ctypes.POINTER(ctypes.c_double)), ctypes.POINTER(i32), ctypes.POINTER(vp),
        ctypes.POINTER(i64), vp]
    for name in EXPORTED_SYMBOLS:
        fn = getattr(lib, name)
        if name not in ("soap_last_error",):
            fn.restype = ctypes.c_int
    _lib = lib
    return lib


# ------------------------------------------------------------------------------------------------
# Python-side views of the C structs
# ------------------------------------------------------------------------------------------------
@dataclass
class Spectra:
    """soap_spectra: `data` is a DEVICE tensor [n_mu, pitch] (or a HOST array/tensor for soap_synthesize_host)."""
    data: object
    n_pix: int
    lambda0: float
    dlambda: float
    contrast: object = None
    lb: Tuple[float, float, float] = (1.0, 0.0, 0.0)

    @property
    def pitch(self) -> int:
        return int(self.data.shape[1])

    def _c(self) -> c_spectra:
        dt = _dtype_code(self.data)
        return c_spectra(_ptr(self.data), int(self.n_pix), self.pitch, dt, float(self.lambda0), float(self.dlambda),
                         _ptr(self.contrast) if self.contrast is not None else None,
                         float(self.lb[0]), float(self.lb[1]), float(self.lb[2]))


def _dtype_code(a) -> int:
    dt = a.dtype
    if dt in (torch.float32, np.dtype(np.float32)):
        return SOAP_F32
    if dt in (torch.float64, np.dtype(np.float64)):
        return SOAP_F64
    raise TypeError(f"unsupported dtype {dt}")


def _ptr(a) -> int:
    if isinstance(a, torch.Tensor):
        return a.data_ptr()
    return a.ctypes.data


def _stream_handle(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream or None
    return int(stream) or None


class Star:
    """Owns one soap_star handle."""

    def __init__(self, device: int = 0):
        self._lib = load_library()
        h = ctypes.c_void_p()
        rc = self._lib.soap_create(ctypes.byref(h), int(device))
        if rc != SOAP_OK:
            raise SoapError(rc, self._lib.soap_last_error(None).decode())
        self._h = h
        self.device = int(device)
        self._keep = None

    def close(self):
        if getattr(self, "_h", None):
            self._lib.soap_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != SOAP_OK:
            raise SoapError(rc, self._lib.soap_last_error(self._h).decode())


def soap_create(device: int = 0) -> Star:
    return Star(device)


def soap_destroy(star: Star) -> None:
    star.close()


def soap_set_option(star: Star, option: int, value: int) -> None:
    star._check(star._lib.soap_set_option(star._h, int(option), int(value)))


def _params(p):
    mu = np.ascontiguousarray(np.asarray(p.mu_centres, dtype=np.float64))
    c = c_star_params(int(p.grid_n), float(p.vsini_kms), float(p.incl_deg), float(p.ld_u1), float(p.ld_u2),
                      int(mu.shape[0]), mu.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                      int(getattr(p, "doppler_mode", 0)), float(getattr(p, "diff_rot", 0.0)))
    return c, mu


def soap_disk_geometry(star: Star, params, stream=None, want_info: bool = True) -> Optional[dict]:
    """params: any object with grid_n, vsini_kms, incl_deg, ld_u1, ld_u2, mu_centres[, doppler_mode]."""
    c, _mu = _params(params)
    info = c_geom_info()
    star._check(star._lib.soap_disk_geometry(star._h, ctypes.byref(c), _stream_handle(stream),
                                             ctypes.byref(info) if want_info else None))
    if not want_info:
        return None
    return dict(n_visible=int(info.n_visible), n_entries=int(info.n_entries), sum_weights=float(info.sum_weights),
                max_abs_dshift=float(info.max_abs_dshift))


def soap_integrate_quiet(star: Star, quiet: Spectra, out: torch.Tensor, stream=None) -> None:
    cq = quiet._c()
    star._check(star._lib.soap_integrate_quiet(star._h, ctypes.byref(cq), out.data_ptr(), _stream_handle(stream)))


def soap_integrate_quiet_static(star: Star, quiet: Spectra, out: torch.Tensor, stream=None) -> None:
    """soap_integrate_quiet for callers that must not allocate device memory: the partial sums go to a fixed 4 MiB
    array inside the library (n_pix <= 524 288; calls that overlap on the GPU race on it) - include/soap_b200.h."""
    cq = quiet._c()
    star._check(star._lib.soap_integrate_quiet_static(star._h, ctypes.byref(cq), out.data_ptr(), _stream_handle(stream)))


def _regions(regions: Sequence):
    arr = (c_region * max(1, len(regions)))()
    for n, (lat, lon, rad, typ) in enumerate(regions):
        arr[n] = c_region(float(lat), float(lon), float(rad), int(typ))
    return arr


def soap_active_timeseries(star: Star, quiet: Spectra, spot: Optional[Spectra], facula: Optional[Spectra],
                           regions: Sequence, phases, out_delta: torch.Tensor, want_n_active: bool = False,
                           stream=None) -> Optional[np.ndarray]:
    """out_delta: DEVICE tensor [n_phases, out_pitch].  Returns n_active (host) if asked (synchronous)."""
    cq = quiet._c()
    cs = spot._c() if spot is not None else None
    cf = facula._c() if facula is not None else None
    ph = np.ascontiguousarray(np.asarray(phases, dtype=np.float64))
    n_ph = int(ph.shape[0])
    na = np.zeros(max(1, n_ph), dtype=np.int32) if want_n_active else None
    out_pitch = int(out_delta.shape[1]) if out_delta.dim() == 2 else int(quiet.n_pix)
    star._check(star._lib.soap_active_timeseries(
        star._h, ctypes.byref(cq), ctypes.byref(cs) if cs is not None else None,
        ctypes.byref(cf) if cf is not None else None, _regions(regions), len(regions),
        ph.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), n_ph, out_delta.data_ptr(), out_pitch,
        na.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)) if na is not None else None, _stream_handle(stream)))
    return na[:n_ph] if na is not None else None


def soap_active_timeseries_effects(star: Star, quiet: Spectra, spot: Optional[Spectra], facula: Optional[Spectra],
                                   regions: Sequence, phases, out_total: Optional[torch.Tensor] = None,
                                   out_flux: Optional[torch.Tensor] = None, out_cb: Optional[torch.Tensor] = None,
                                   want_n_active: bool = False, stream=None) -> Optional[np.ndarray]:
    """Total / flux-only / CB-only delta spectra (Eq. 1-3); each output a DEVICE tensor [n_phases, out_pitch] or None."""
    cq = quiet._c()
    cs = spot._c() if spot is not None else None
    cf = facula._c() if facula is not None else None
    ph = np.ascontiguousarray(np.asarray(phases, dtype=np.float64))
    n_ph = int(ph.shape[0])
    na = np.zeros(max(1, n_ph), dtype=np.int32) if want_n_active else None
    outs = [o for o in (out_total, out_flux, out_cb) if o is not None]
    pitches = {int(o.shape[1]) for o in outs}
    if len(pitches) > 1:
        raise ValueError("outputs must share one pitch")
    out_pitch = pitches.pop() if pitches else int(quiet.n_pix)
    star._check(star._lib.soap_active_timeseries_effects(
        star._h, ctypes.byref(cq), ctypes.byref(cs) if cs is not None else None,
        ctypes.byref(cf) if cf is not None else None, _regions(regions), len(regions),
        ph.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), n_ph,
        out_total.data_ptr() if out_total is not None else None, out_flux.data_ptr() if out_flux is not None else None,
        out_cb.data_ptr() if out_cb is not None else None, out_pitch,
        na.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)) if na is not None else None, _stream_handle(stream)))
    return na[:n_ph] if na is not None else None


def soap_active_timeseries_evolving(star: Star, quiet: Spectra, spot: Optional[Spectra], facula: Optional[Spectra],
                                    regions: Sequence, phases, radii, out_total: Optional[torch.Tensor] = None,
                                    out_flux: Optional[torch.Tensor] = None, out_cb: Optional[torch.Tensor] = None,
                                    want_n_active: bool = False, stream=None) -> Optional[np.ndarray]:
    """As soap_active_timeseries_effects with radii[n_phases, n_regions] (HOST): evolving regions, <= 0 = absent."""
    cq = quiet._c()
    cs = spot._c() if spot is not None else None
    cf = facula._c() if facula is not None else None
    ph = np.ascontiguousarray(np.asarray(phases, dtype=np.float64))
    n_ph = int(ph.shape[0])
    rr = np.ascontiguousarray(np.asarray(radii, dtype=np.float64)).reshape(n_ph, len(regions))
    na = np.zeros(max(1, n_ph), dtype=np.int32) if want_n_active else None
    outs = [o for o in (out_total, out_flux, out_cb) if o is not None]
    out_pitch = int(outs[0].shape[1]) if outs else int(quiet.n_pix)
    star._check(star._lib.soap_active_timeseries_evolving(
        star._h, ctypes.byref(cq), ctypes.byref(cs) if cs is not None else None,
        ctypes.byref(cf) if cf is not None else None, _regions(regions), len(regions),
        ph.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), n_ph, rr.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
        out_total.data_ptr() if out_total is not None else None, out_flux.data_ptr() if out_flux is not None else None,
        out_cb.data_ptr() if out_cb is not None else None, out_pitch,
        na.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)) if na is not None else None, _stream_handle(stream)))
    return na[:n_ph] if na is not None else None


def soap_contrast_planck(star: Star, lambda0: float, dlambda: float, n_pix: int, t_quiet: float, t_active: float,
                         out: torch.Tensor, stream=None) -> torch.Tensor:
    """SOAPcontrast: out[m] = B_lambda(t_active) / B_lambda(t_quiet), lambda in Angstrom; out: DEVICE [n_pix]."""
    if not out.is_contiguous() or out.numel() < n_pix:
        raise ValueError("out must be a contiguous device tensor of at least n_pix elements")
    star._check(star._lib.soap_contrast_planck(star._h, float(lambda0), float(dlambda), int(n_pix), float(t_quiet), float(t_active),
                                               out.data_ptr(), _dtype_code(out), _stream_handle(stream)))
    return out


def soap_line_rvs(star: Star, rows: torch.Tensor, n_pix: int, lambda0: float, dlambda: float, centres: torch.Tensor,
                  half_widths: torch.Tensor, norm: torch.Tensor, edge: int = 0, stream=None) -> torch.Tensor:
    """First-moment RV (cm/s) of every line in every row; all tensors on the device, centres / half_widths / norm fp64."""
    r2 = rows if rows.dim() == 2 else rows.unsqueeze(0)
    for t in (centres, half_widths, norm):
        if t.dtype != torch.float64 or not t.is_contiguous():
            raise ValueError("centres, half_widths and norm must be contiguous fp64 device tensors")
    out = torch.empty((r2.shape[0], centres.shape[0]), dtype=torch.float64, device=rows.device)
    star._check(star._lib.soap_line_rvs(
        star._h, r2.data_ptr(), int(r2.shape[0]), int(n_pix), int(r2.stride(0)), _dtype_code(r2), float(lambda0), float(dlambda),
        centres.data_ptr(), half_widths.data_ptr(), int(centres.shape[0]), norm.data_ptr(), int(edge), out.data_ptr(),
        _stream_handle(stream)))
    return out


def soap_lower_resolution(star: Star, rows: torch.Tensor, n_pix: int, lambda0: float, dlambda: float, resolution: float,
                          out: torch.Tensor, stream=None) -> None:
    """rows, out: DEVICE tensors [n_rows, pitch] (or [pitch]) of one dtype; Gaussian LSF of FWHM lambda/resolution."""
    r2 = rows if rows.dim() == 2 else rows.unsqueeze(0)
    o2 = out if out.dim() == 2 else out.unsqueeze(0)
    if r2.dtype != o2.dtype or r2.shape[0] != o2.shape[0]:
        raise ValueError("rows and out must agree in dtype and row count")
    star._check(star._lib.soap_lower_resolution(
        star._h, r2.data_ptr(), int(r2.shape[0]), int(n_pix), int(r2.stride(0)), _dtype_code(r2), float(lambda0),
        float(dlambda), float(resolution), o2.data_ptr(), int(o2.stride(0)), _stream_handle(stream)))


def soap_export_geometry(star: Star, grid_n: int) -> dict:
    n = grid_n * grid_n
    mu, vel, w = (np.zeros(n, dtype=np.float64) for _ in range(3))
    b = np.zeros(n, dtype=np.int32)
    star._check(star._lib.soap_export_geometry(star._h, mu.ctypes.data, vel.ctypes.data, w.ctypes.data, b.ctypes.data))
    return dict(mu=mu, vel=vel, w=w, bin=b)


def soap_get_stats(star: Star, stream=None) -> dict:
    st = c_stats()
    star._check(star._lib.soap_get_stats(star._h, ctypes.byref(st), _stream_handle(stream)))
    return {k: (float(getattr(st, k)) if k.endswith('_ms') else int(getattr(st, k))) for k, _ in c_stats._fields_}


def soap_synthesize_host(star: Star, params, quiet: Spectra, spot: Optional[Spectra], facula: Optional[Spectra],
                         regions: Sequence, phases, out_quiet, out_delta, want_n_active: bool = False, stream=None):
    """All Spectra.data / contrast, out_quiet [n_pix] and out_delta [n_phases, n_pix] are HOST arrays
    (numpy, or CPU torch tensors - pinned for full copy bandwidth)."""
    c, _mu = _params(params)
    cq = quiet._c()
    cs = spot._c() if spot is not None else None
    cf = facula._c() if facula is not None else None
    ph = np.ascontiguousarray(np.asarray(phases, dtype=np.float64))
    n_ph = int(ph.shape[0])
    na = np.zeros(max(1, n_ph), dtype=np.int32) if want_n_active else None
    star._check(star._lib.soap_synthesize_host(
        star._h, ctypes.byref(c), ctypes.byref(cq), ctypes.byref(cs) if cs is not None else None,
        ctypes.byref(cf) if cf is not None else None, _regions(regions), len(regions),
        ph.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), n_ph, _ptr(out_quiet),
        _ptr(out_delta) if out_delta is not None else None,
        na.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)) if na is not None else None, _stream_handle(stream)))
    return na[:n_ph] if na is not None else None


def soap_batch_disk_geometry(stars: Sequence[Star], params: Sequence, stream=None, want_info: bool = False):
    """The geometry of many stars in one launch; params[k] as for soap_disk_geometry.  Returns a list of info dicts or None."""
    n = len(stars)
    lib = stars[0]._lib
    hs = (ctypes.c_void_p * n)(*[s._h for s in stars])
    cps = [_params(p) for p in params]  # (struct, mu array kept alive)
    pp = (ctypes.POINTER(c_star_params) * n)(*[ctypes.pointer(c) for c, _ in cps])
    infos = (c_geom_info * n)() if want_info else None
    rc = lib.soap_batch_disk_geometry(hs, n, pp, _stream_handle(stream), infos)
    if rc != SOAP_OK:
        msgs = [lib.soap_last_error(s._h).decode() for s in stars]
        raise SoapError(rc, "; ".join(m for m in msgs if m))
    if not want_info:
        return None
    return [dict(n_visible=int(i.n_visible), n_entries=int(i.n_entries), sum_weights=float(i.sum_weights),
                 max_abs_dshift=float(i.max_abs_dshift)) for i in infos]


def soap_batch_integrate_quiet(stars: Sequence[Star], quiet: Sequence[Spectra], out: Sequence[torch.Tensor],
                               stream=None) -> None:
    n = len(stars)
    lib = stars[0]._lib
    hs = (ctypes.c_void_p * n)(*[s._h for s in stars])
    cqs = [q._c() for q in quiet]
    qp = (ctypes.POINTER(c_spectra) * n)(*[ctypes.pointer(c) for c in cqs])
    op = (ctypes.c_void_p * n)(*[o.data_ptr() for o in out])
    rc = lib.soap_batch_integrate_quiet(hs, n, qp, op, _stream_handle(stream))
    if rc != SOAP_OK:
        msgs = [lib.soap_last_error(s._h).decode() for s in stars]
        raise SoapError(rc, "; ".join(m for m in msgs if m))


def soap_batch_active_timeseries(stars: Sequence[Star], quiet: Sequence[Spectra], spot: Sequence[Optional[Spectra]],
                                 facula: Sequence[Optional[Spectra]], regions: Sequence[Sequence],
                                 phases: Sequence, out_delta: Sequence[torch.Tensor], stream=None) -> None:
    n = len(stars)
    lib = stars[0]._lib
    hs = (ctypes.c_void_p * n)(*[s._h for s in stars])
    keep = []

    def parr(specs):
        cs = [(s._c() if s is not None else None) for s in specs]
        keep.append(cs)
        return (ctypes.POINTER(c_spectra) * n)(*[(ctypes.pointer(c) if c is not None else None) for c in cs])

    qp, sp, fp = parr(quiet), parr(spot), parr(facula)
    regs = [_regions(r) for r in regions]
    rp = (ctypes.POINTER(c_region) * n)(*[ctypes.cast(r, ctypes.POINTER(c_region)) for r in regs])
    nr = (ctypes.c_int32 * n)(*[len(r) for r in regions])
    phs = [np.ascontiguousarray(np.asarray(p, dtype=np.float64)) for p in phases]
    pp = (ctypes.POINTER(ctypes.c_double) * n)(*[p.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) for p in phs])
    nph = (ctypes.c_int32 * n)(*[int(p.shape[0]) for p in phs])
    op = (ctypes.c_void_p * n)(*[o.data_ptr() for o in out_delta])
    pitch = (ctypes.c_int64 * n)(*[int(o.shape[1]) for o in out_delta])
    rc = lib.soap_batch_active_timeseries(hs, n, qp, sp, fp, rp, nr, pp, nph, op, pitch, _stream_handle(stream))
    if rc != SOAP_OK:
        msgs = [lib.soap_last_error(s._h).decode() for s in stars]
        raise SoapError(rc, "; ".join(m for m in msgs if m))


# ------------------------------------------------------------------------------------------------
# marshalling helper: numpy workload arrays -> device Spectra (pitch padded to a multiple of 4)
# ------------------------------------------------------------------------------------------------
def to_device_spectra(rows: np.ndarray, lambda0: float, dlambda: float, device, contrast: Optional[np.ndarray] = None,
                      lb=(1.0, 0.0, 0.0)) -> Spectra:
    rows = np.asarray(rows)
    n_mu, n_pix = rows.shape
    pitch = (n_pix + 3) & ~3
    tdt = torch.float32 if rows.dtype == np.float32 else torch.float64
    data = torch.zeros((n_mu, pitch), dtype=tdt, device=device)
    data[:, :n_pix] = torch.from_numpy(np.ascontiguousarray(rows)).to(device)
    c = None
    if contrast is not None:
        c = torch.from_numpy(np.ascontiguousarray(np.asarray(contrast, dtype=rows.dtype))).to(device)
    return Spectra(data=data, n_pix=n_pix, lambda0=lambda0, dlambda=dlambda, contrast=c, lb=tuple(lb))
