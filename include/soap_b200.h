/*
 * soap_b200.h - C ABI of the B200-native SOAP disk-integration hot path.
 *
 * What the library computes (Zhao & Dumusque 2023, "SOAP-GPU", arXiv:2301.04259; "P:n" = line n of
 * PAPER.md, "S#" = a reading listed in DESIGN.md section 3):
 *
 *   A star is an N x N grid of cells over [-1,1]^2.  Every visible cell carries a rotational
 *   velocity and a limb-darkening intensity (Fig. 1).  The cell's local spectrum - the row of a
 *   mu-binned spectrum table whose mu is closest to the cell's - is Doppler-shifted by the
 *   cell's velocity and linearly interpolated back onto the uniform wavelength grid (Eq. 5-9,
 *   P:160-186), weighted, and summed over cells: once for the quiet star (Alg. 1) and, for
 *   every rotational phase, over the cells covered by active regions only (InfoMap, Alg. 5)
 *   to give the active-minus-quiet delta spectrum (Eq. 3-4).
 *
 * Conventions common to every entry point
 *   - Every function returns an int status: SOAP_OK (0) or a negative soap_status.  Nothing throws or
 *     aborts across the ABI.  Argument errors are detected before any device write (no partial output).
 *   - "DEVICE" pointers are CUDA device pointers on the device the handle was created for; "HOST"
 *     pointers are ordinary host memory.  The caller owns every input and output buffer.  The library
 *     owns only what lives inside soap_star (geometry, binned weights, scratch, active-entry lists) and
 *     frees it in soap_destroy.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All device work
 *     is enqueued on it; a call is asynchronous unless it has a non-NULL HOST output pointer
 *     (`info`, `n_active`, export, stats), in which case it synchronises that stream before returning.
 *     Scratch is (re)allocated with cudaMalloc when a call needs more than any earlier call did; once
 *     sizes have been seen, calls allocate nothing.  A single star's soap_active_timeseries* call passes its
 *     region centres as kernel arguments (up to 192 (phase, region) pairs) and copies nothing; larger calls
 *     and the batch calls stage them through a ring of pinned host buffers guarded by events and must not be
 *     stream-captured.  A single star's geometry / quiet / time-series calls with HOST outputs NULL, after one
 *     un-captured call of the same sizes (scratch allocated), enqueue kernels only and CAN be captured in a
 *     CUDA graph (tests/test_gpu_edges.py); the captured step is fixed: its regions and phases are kernel
 *     arguments of the graph's nodes.
 *   - The launches of a handle's consecutive calls on one stream (geometry, quiet, active map, active delta)
 *     are chained with programmatic dependent launch: a launch may start while its predecessor drains and
 *     waits on the device before it reads what the predecessor wrote.  Nothing changes for the caller.
 *   - A handle is not re-entrant: calls on one soap_star must not run concurrently (from several host
 *     threads or on several streams at once) - its scratch, its self-resetting device counters and its
 *     staging ring belong to one call at a time.  Different handles are independent.
 *   - There is no CPU fallback and no other backend: without a CUDA device every compute entry point
 *     returns SOAP_ERR_CUDA.
 *   - Cell indexing: c = j * N + i with j the column (x) index and i the row (y) index;
 *     x_j = -1 + (2j+1)/N, y_i = -1 + (2i+1)/N (S1).
 *   - Results are run-to-run bit-identical (no unordered floating-point atomics).
 */
#ifndef SOAP_B200_H
#define SOAP_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SOAP_B200_VERSION 100 /* major*100 + minor */

typedef struct soap_star soap_star; /* opaque; one star's device-resident state */

enum soap_status {
    SOAP_OK = 0,
    SOAP_ERR_INVALID_ARG = -1, /* bad pointer / size / flag; nothing was written */
    SOAP_ERR_NOT_READY = -2,   /* soap_disk_geometry has not been called on this handle */
    SOAP_ERR_CUDA = -3,        /* a CUDA runtime call failed (see soap_last_error) */
    SOAP_ERR_OOM = -4,         /* device or host allocation failed */
    SOAP_ERR_UNSUPPORTED = -5  /* valid request this build does not implement */
};

enum soap_dtype { SOAP_F32 = 0, SOAP_F64 = 1 };
enum soap_region_type { SOAP_SPOT = 1, SOAP_FACULA = 2 };
/* The three per-cell differences of PAPER.md:73-79, with this library's sign (active minus quiet). */
enum soap_effect { SOAP_EFFECT_TOTAL = 0, SOAP_EFFECT_FLUX = 1, SOAP_EFFECT_CB = 2 };

/* How the shift-interpolate-accumulate sum is evaluated.  All forms compute the same sums (Alg. 1,
 * Eq. 3) and differ only in rounding order. */
enum soap_form {
    SOAP_FORM_AUTO = 0,   /* library picks.  Solid-body rotation: SOAP_FORM_COMPOSITE (quiet spectrum of fp32 tables with
                             n_mu <= 24; binned entries for everything else).  Differential rotation (diff_rot != 0):
                             one entry per cell with the run collapse of SOAP_FORM_FIR */
    SOAP_FORM_BINNED = 1, /* cells pre-binned by (column, mu-bin): all cells of a column share one
                             velocity under solid-body rotation (BASELINE.json north_star) */
    SOAP_FORM_CELLS = 2,  /* one entry per visible cell - the literal double loop of Alg. 1 */
    SOAP_FORM_FIR = 3,    /* binned (or, under differential rotation, per-cell) entries; per wavelength tile every
                             run of entries of one spectrum row with the same integer shift is collapsed into one
                             record {sum W, sum W a}: taps linear in the pixel index (exact in exact arithmetic) */
    SOAP_FORM_COMPOSITE = 4 /* binned weights; quiet spectrum: per column j the composite T_j = sum_b W[j,b] S_b is formed
                             from unshifted samples (1 FMA per (column, mu-bin, pixel)) and interpolated once per
                             (column, pixel) - lerp is linear in the spectrum and the cells of a column share one
                             velocity.  Cost independent of v sin i.  fp32 spectra, solid body, n_mu <= 24; otherwise
                             (and for the active delta spectra) the binned entries are used */
};

enum soap_option {
    SOAP_OPT_FORM = 1,         /* value: enum soap_form; default SOAP_FORM_AUTO */
    SOAP_OPT_QUIET_SPLITS = 2, /* value: >0 forces the number of entry-chunks the quiet sum is split
                                  into across CTAs; 0 (default) = sized from the SM count */
    SOAP_OPT_KERNEL_TIMING = 3, /* value: 1 brackets the shift-interpolate-accumulate kernel of each call with
                                  CUDA events on the caller's stream; soap_get_stats reports the durations */
    SOAP_OPT_EFFECT_PASSES = 4 /* value: 1 makes soap_active_timeseries_effects / _evolving run one pass per
                                  requested effect; 0 (default): two or three effects come from one pass */
};

/* Star / disk description.  HOST, read only during the call. */
typedef struct {
    int32_t grid_n;           /* N >= 1 */
    double vsini_kms;         /* v_cell = x * vsini_kms * sin(incl)  (S5; +x is the receding limb) */
    double incl_deg;          /* angle between spin axis and line of sight (S13) */
    double ld_u1, ld_u2;      /* quadratic limb darkening: w = 1 - u1 (1-mu) - u2 (1-mu)^2  (S3, S4) */
    int32_t n_mu;             /* number of mu bins, 1..SOAP_MAX_MU */
    const double *mu_centres; /* HOST [n_mu], strictly ascending (S9: nearest centre, tie -> larger mu) */
    int32_t doppler_mode;     /* 0: relativistic, Eq. 6 (source wavelength lambda * sqrt((1-b)/(1+b)));
                                 1: first order, lambda * (1 - v/c)  (S6) */
    double diff_rot;          /* differential rotation omega_1 / omega_0 of omega = omega_0 + omega_1 sin^2(latitude)
                                 (-0.18 for the Sun); v_cell is multiplied by 1 + diff_rot sin^2(latitude).
                                 0 = solid body.  Non-zero selects the per-cell form (R-DR); must be > -1. */
} soap_star_params;

#define SOAP_MAX_MU 64

/* One table of mu-binned spectra on the uniform grid lambda_m = lambda0 + m * dlambda (Eq. 5). */
typedef struct {
    const void *data;         /* DEVICE [n_mu][pitch] row-major, n_pix valid values per row,
                                 base address 16-byte aligned */
    int64_t n_pix;            /* P >= 2 */
    int64_t pitch;            /* row pitch in elements, >= n_pix, multiple of 4 */
    int32_t dtype;            /* enum soap_dtype; outputs use the same dtype */
    double lambda0, dlambda;  /* dlambda > 0, lambda0 > 0 */
    const void *contrast;     /* DEVICE [n_pix] of `dtype`, or NULL (== 1).  I_ratio of Eq. 3, applied
                                 at the output pixel after the shift (S17).  Ignored for quiet. */
    double lb_c0, lb_c1, lb_c2; /* LB(mu) = c0 + c1 mu + c2 mu^2, per cell with its exact mu (Eq. 11-12,
                                   P:372-379).  Ignored for quiet; (1,0,0) for spots. */
} soap_spectra;

typedef struct {
    double lat_deg, lon_deg;  /* region centre; effective longitude = lon + 360 * phase, 0 = sub-observer
                                 meridian, increasing toward +x (S12) */
    double radius;            /* in stellar radii, 0 < radius < 1: radius of the circle the region projects
                                 to at disk centre; angular radius asin(radius) (S11) */
    int32_t type;             /* enum soap_region_type */
} soap_region;

typedef struct {
    int64_t n_visible;        /* cells whose centre lies on the disk (S2) */
    int64_t n_entries;        /* (column, mu-bin) pairs with non-zero weight (n_visible for FORM_CELLS) */
    double sum_weights;       /* sum of w over visible cells: the integrated continuum of a unit spectrum (S4) */
    double max_abs_dshift;    /* max |D - 1| over cells; |shift in pixels| <= this * (lambda0/dlambda + P) */
} soap_geom_info;

typedef struct {
    int64_t quiet_entries;        /* entries summed per pixel by the last soap_integrate_quiet */
    int64_t active_entries;       /* sum over phases of (row, column) entries of the last time series,
                                     counting the quiet-row and the active-row entry of a pair separately */
    int64_t active_cells;         /* sum over phases of covered cells */
    int32_t quiet_splits, tile_px;
    int32_t form;                 /* enum soap_form the last soap_integrate_quiet actually ran (the form selected by
                                     soap_disk_geometry when no quiet spectrum has been computed yet) */
    int32_t launches;             /* kernels launched by this handle since soap_create */
    float quiet_kernel_ms;        /* SOAP_OPT_KERNEL_TIMING: device time of the last quiet / active */
    float active_kernel_ms;       /*   shift-interpolate-accumulate kernel launch; else 0 */
} soap_stats;

/* ---- lifetime ---------------------------------------------------------------------------------- */
int soap_version(void);
/* Create an empty handle bound to CUDA device `device`.  *out is set to NULL on failure. */
int soap_create(soap_star **out, int device);
/* Frees all device and host memory of the handle.  NULL is allowed. */
int soap_destroy(soap_star *star);
/* Library-owned, NUL-terminated description of the last error on this handle (valid until the next
 * call on it).  star == NULL returns the message of the last failed soap_create. */
const char *soap_last_error(const soap_star *star);
int soap_set_option(soap_star *star, int32_t option, int64_t value);
/* Copies counters of the last calls to HOST *stats; synchronises `stream`. */
int soap_get_stats(soap_star *star, soap_stats *stats, void *stream);

/* ---- a1 + a2: geometry and (column, mu-bin) weight binning (S1-S5, S9, S10) ----------------
 * Computes, on the device, every cell's (x, y, mu, v, w, bin), the per-column Doppler shift factor
 * D_j - 1 in fp64, and the binned weights W[j,b] = sum of w over the cells of column j in bin b.
 * `info` (HOST, nullable) receives the summary; non-NULL makes the call synchronous. */
int soap_disk_geometry(soap_star *star, const soap_star_params *params, void *stream, soap_geom_info *info);

/* ---- a3: quiet integrated spectrum (Alg. 1) ---------------------------------------------
 * out[m] = sum over visible cells of w_c * lerp(S_quiet[bin_c]; source coordinate of pixel m under D_c),
 * clamped to the end values outside the grid (S8).  `out`: DEVICE [n_pix] of quiet->dtype. */
int soap_integrate_quiet(soap_star *star, const soap_spectra *quiet, void *out, void *stream);

/* ---- a3 for callers that must not allocate device memory (Alg. 1) ------------------------
 * The same sum as soap_integrate_quiet, same arguments, fp32 or fp64 tables, any rotation law - but this call never
 * allocates or frees device memory, on any call, whatever the sizes.  It is meant for programs in which the library may
 * not go to the CUDA allocator once they are running: an application that has given the whole device to its own memory
 * pool, so that a cudaMalloc here would fail; or a service loop that cannot take the device-wide synchronisation a
 * cudaMalloc / cudaFree brings.  Create the handle and call soap_disk_geometry during set-up (those do allocate); from
 * then on this entry point only enqueues two kernels on `stream`.
 *   Scratch: the fp64 partial sums of the entry chunks live in a 4 MiB array that is part of the library image
 *     (every device that loads the library holds it until the process exits).  The limit that follows:
 *     round_up4(n_pix) <= 524 288, else SOAP_ERR_UNSUPPORTED with a message naming the limit and nothing is written.
 *     Within the limit the entry list is cut into fewer chunks when the array cannot hold as many as
 *     soap_integrate_quiet would take, so long spectra run with less parallelism over entries.
 *   First call on a device: looks up the array's device address (once per device, with that device current).  Make
 *     that first call during set-up, before any stream capture is under way in the process.
 *   Sharing: every call on a device, from every handle, uses the one array.  Each call overwrites what it later reads,
 *     so nothing left by an earlier call matters; but two calls whose kernels overlap on the GPU (different streams,
 *     no dependency between them) race on it and give wrong spectra.  Order them on one stream or with events.
 *   Result: the direct (binned or per-cell) form with fp64 chunk sums added in chunk order; equal to
 *     soap_integrate_quiet to rounding (bit-identical for fp64 tables when both take the same number of chunks).
 *   SOAP_OPT_QUIET_SPLITS is honoured up to what the array holds; SOAP_OPT_KERNEL_TIMING and soap_get_stats' quiet
 *     fields are not updated by this call. */
int soap_integrate_quiet_static(soap_star *star, const soap_spectra *quiet, void *out, void *stream);

/* ---- a4 + a5 + a6: active-region delta spectra for every phase (Alg. 5, Eq. 3; S11-S19) ----------
 * For phase p: type[c] = type of the LAST region in list order covering visible cell c, and
 *   out_delta[p][m] = sum over covered cells of
 *        w_c * ( C_t[m] * LB_t(mu_c) * lerp(S_t[bin_c]; c, m)  -  lerp(S_quiet[bin_c]; c, m) )
 * i.e. active minus quiet (the negative of Eq. 3), so that S_final = S_quiet,integrated + delta (Eq. 4).
 * Phases without covered cells give exact zeros.
 *   spot / facula: nullable if no region of that type is listed; must match quiet in n_pix, pitch
 *                  rules, dtype, lambda0, dlambda.
 *   regions: HOST [n_regions] (n_regions may be 0);  phases: HOST [n_phases], in rotations, any real.
 *   out_delta: DEVICE [n_phases][out_pitch] of quiet->dtype, out_pitch >= n_pix.
 *   n_active: HOST [n_phases] or NULL; number of covered cells per phase (non-NULL => synchronous). */
int soap_active_timeseries(soap_star *star, const soap_spectra *quiet, const soap_spectra *spot,
                           const soap_spectra *facula, const soap_region *regions, int32_t n_regions,
                           const double *phases, int32_t n_phases, void *out_delta, int64_t out_pitch,
                           int32_t *n_active, void *stream);

/* ---- flux-only and convective-blueshift-only time series beside the total (Eq. 1-3) -----
 * Same arguments, covered cells and conventions as soap_active_timeseries; I_ratio = C_t[m] LB_t(mu_c):
 *   out_total[p][m] = sum w_c ( I_ratio lerp(S_t[bin_c]) - lerp(S_quiet[bin_c]) )     (negative of Eq. 3)
 *   out_flux [p][m] = sum w_c ( I_ratio lerp(S_quiet[bin_c]) - lerp(S_quiet[bin_c]) ) (negative of Eq. 1)
 *   out_cb   [p][m] = sum w_c (         lerp(S_t[bin_c]) - lerp(S_quiet[bin_c]) )     (negative of Eq. 2)
 * Each output: DEVICE [n_phases][out_pitch] or NULL (that effect is skipped); at least one non-NULL.
 * fp32 spectra, solid-body rotation, two or three outputs requested: ONE active map and ONE
 * shift-interpolate-accumulate launch (2 launches per call) - the outputs are three weightings of the same
 * interpolated sums, kept apart per region type: the cost of the total alone when both limb-brightening laws
 * are 1, and the entries of a type with a law other than 1 are walked twice (weights w and w LB_t).  Results
 * agree with the pass-per-effect form to rounding (not bit for bit; each form is run-to-run identical).
 * Otherwise (one output, fp64 spectra, differential rotation, SOAP_OPT_EFFECT_PASSES = 1): one launch per
 * requested effect; the active map is built once for total and flux, and once more for CB only when a
 * limb-brightening law differs from 1. */
int soap_active_timeseries_effects(soap_star *star, const soap_spectra *quiet, const soap_spectra *spot,
                                   const soap_spectra *facula, const soap_region *regions, int32_t n_regions,
                                   const double *phases, int32_t n_phases, void *out_total, void *out_flux,
                                   void *out_cb, int64_t out_pitch, int32_t *n_active, void *stream);

/* ---- evolving regions: the same three outputs with a radius per (phase, region) -----------
 * radii: HOST [n_phases][n_regions], the radius (same convention as soap_region.radius) of region r at phase p;
 * a value <= 0 means the region is absent at that phase; every value must be < 1.  NULL = regions[r].radius.
 * The evolution law itself (linear growth / decay, asymmetric Gaussian) is the caller's: it is input preparation. */
int soap_active_timeseries_evolving(soap_star *star, const soap_spectra *quiet, const soap_spectra *spot,
                                    const soap_spectra *facula, const soap_region *regions, int32_t n_regions,
                                    const double *phases, int32_t n_phases, const double *radii, void *out_total,
                                    void *out_flux, void *out_cb, int64_t out_pitch, int32_t *n_active, void *stream);

/* ---- resolution lowering (Alg. 2, Alg. 5) ------------------------------------
 * "Lower the resolution of the final spectrum to match the resolution provided in the configuration file."  The
 * paper names no kernel; this library's reading (DESIGN.md R-LSF) is a Gaussian line-spread function of FWHM
 * lambda / resolution, sampled on the pixel grid and normalised at every output pixel, truncated at 5 sigma, ends
 * clamped (S8):  out[r][m] = sum_j g_m(j) in[r][clamp(m+j)] / sum_j g_m(j),  g_m(j) = exp(-(j dlambda)^2 / 2 sigma_m^2),
 * sigma_m = lambda_m / (resolution * 2 sqrt(2 ln 2)).  Rows are independent (e.g. Q + delta_p for every phase).
 *   in:  DEVICE [n_rows][in_pitch] of `dtype`;  out: DEVICE [n_rows][out_pitch], must not alias `in`.
 * Needs no geometry.  SOAP_ERR_UNSUPPORTED if the LSF is wider than 96 pixels on a side. */
int soap_lower_resolution(soap_star *star, const void *in, int64_t n_rows, int64_t n_pix, int64_t in_pitch,
                          int32_t dtype, double lambda0, double dlambda, double resolution, void *out,
                          int64_t out_pitch, void *stream);

/* ---- SOAPcontrast: wavelength-dependent contrast of an active region modelled by a temperature ----
 * "Derives the contrast by calculating the ratio of two Planck functions at two different effective temperatures", one
 * value per wavelength pixel:
 *   out[m] = B_lambda(t_active) / B_lambda(t_quiet),  B_lambda(T) = (2 h c^2 / lambda^5) / (exp(h c / (lambda k_B T)) - 1),
 *   lambda = lambda0 + m dlambda in ANGSTROM; temperatures in Kelvin (> 0).  Evaluated in fp64, rounded once to `dtype`.
 * The result is what soap_spectra.contrast expects (the I_ratio of Eq. 3, applied after the shift, S17).
 *   out: DEVICE [n_pix] of `dtype`.  Needs no geometry.  Asynchronous on `stream`. */
int soap_contrast_planck(soap_star *star, double lambda0, double dlambda, int64_t n_pix, double t_quiet, double t_active,
                         void *out, int32_t dtype, void *stream);

/* ---- first-moment radial velocity of spectral lines (the RV reduction that follows the path) -----
 * The paper cross-correlates with a mask and fits a Gaussian; the mask is not available, and BASELINE.json's
 * acceptance functional is a first-moment RV per line, which this entry point computes on the device:
 *   window m_lo = ceil((lc - hw - lambda0)/dlambda) .. m_hi = floor((lc + hw - lambda0)/dlambda), depth = 1 - F[r][m]/norm[r],
 *   out_rv[r][l] = c * sum (lambda_m - lc) depth / sum depth / lc   in cm/s;
 *   NaN when the window is not inside [edge, n_pix - edge) or the depths sum to 0.
 * rows: DEVICE [n_rows][pitch] of `dtype`;  centres, half_widths: DEVICE [n_lines] fp64 (Angstrom);
 * norm: DEVICE [n_rows] fp64 (continuum level, e.g. sum_weights);  out_rv: DEVICE [n_rows][n_lines] fp64. */
int soap_line_rvs(soap_star *star, const void *rows, int64_t n_rows, int64_t n_pix, int64_t pitch, int32_t dtype,
                  double lambda0, double dlambda, const double *centres, const double *half_widths, int64_t n_lines,
                  const double *norm, int64_t edge, double *out_rv, void *stream);

/* ---- debug export of the geometry (HOST outputs, N*N each, any may be NULL; synchronous) --------
 * Hidden cells: mu = 0, vel = 0, w = 0, bin = -1. */
int soap_export_geometry(soap_star *star, double *mu, double *vel, double *w, int32_t *bin);

/* ---- end-to-end convenience with HOST buffers ---------------------------------------------------
 * Same computation as soap_disk_geometry + soap_integrate_quiet + soap_active_timeseries, but every
 * spectra / contrast pointer in quiet / spot / facula, `out_quiet` ([n_pix]) and `out_delta`
 * ([n_phases][n_pix], densely packed) are HOST pointers; the library stages the tables through device
 * buffers it owns (the copies are part of the call).  Synchronous.  Long fp32 spectra are processed in a
 * few wavelength chunks so that the upload of one chunk overlaps the kernels of the previous one; when the
 * outputs are pinned (device-visible) host memory the kernels store straight into them, otherwise they are
 * staged and copied back chunk by chunk.  Results equal those of the device-resident calls up to the order
 * of the fp64 partial sums (a few fp32 ulps). */
int soap_synthesize_host(soap_star *star, const soap_star_params *params, const soap_spectra *quiet,
                         const soap_spectra *spot, const soap_spectra *facula, const soap_region *regions,
                         int32_t n_regions, const double *phases, int32_t n_phases, void *out_quiet,
                         void *out_delta, int32_t *n_active, void *stream);

/* ---- config 5: many independent stars in one call ----------------------------------------------
 * Arrays of length n_stars of the arguments above; star k uses stars[k], quiet[k], ...  Every argument of
 * every star is checked before anything is enqueued.  fp32 tables under solid-body rotation (the composite-
 * column form for the quiet spectra) take ONE launch per call for all stars - soap_batch_active_timeseries:
 * one active-map launch (a cluster per (star, phase)) and one shift-interpolate-accumulate launch over the
 * (star, phase, tile) items - enqueued on `stream`; the stars' descriptors are staged in scratch of
 * stars[0], which must therefore outlive the call's device work.  Mixed batches (fp64 tables, differential
 * rotation, several devices) fall back to per-star launches dealt to `stream` and two side streams of
 * stars[0], forked from and joined back into `stream` with events.  A star must not appear twice in a batch;
 * no stream capture. */
/* soap_disk_geometry for n_stars stars in ONE launch (every star's CTAs side by side, each star with its own
 * finalisation).  params: HOST array of n_stars pointers.  infos: HOST [n_stars] or NULL; non-NULL synchronises `stream`.
 * Stars on several devices (or n_stars == 1) are served by per-star calls. */
int soap_batch_disk_geometry(soap_star *const *stars, int32_t n_stars, const soap_star_params *const *params, void *stream,
                             soap_geom_info *infos);
int soap_batch_integrate_quiet(soap_star *const *stars, int32_t n_stars, const soap_spectra *const *quiet,
                               void *const *out, void *stream);
int soap_batch_active_timeseries(soap_star *const *stars, int32_t n_stars, const soap_spectra *const *quiet,
                                 const soap_spectra *const *spot, const soap_spectra *const *facula,
                                 const soap_region *const *regions, const int32_t *n_regions,
                                 const double *const *phases, const int32_t *n_phases,
                                 void *const *out_delta, const int64_t *out_pitch, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* SOAP_B200_H */
