/*
 * soap_oracle.c - TEST INFRASTRUCTURE, not product code.
 *
 * Plain fp64 CPU oracle for the SOAP-GPU disk-integration hot path (Zhao & Dumusque 2023,
 * arXiv:2301.04259; citations "P:n" are line numbers of /root/reference/PAPER.md).
 * It is the *definition* of what the CUDA path must compute, written one cell at a time:
 *
 *   geometry   P:49  (N x N cells, velocity + limb-darkening intensity per cell), Fig. 1
 *   quiet      Alg. 1:  for every cell: shift S_quiet by vel_{X,Y}, linearly interpolate
 *              back onto the grid, weight by I_{X,Y}, accumulate
 *   shift      Eq. 5-9 P:160-186 (uniform grid lambda_n = lambda_0 + n k; Doppler factor of Eq. 6);
 *              written as the equivalent gather (reading S7): S'(lambda_m) is the linear
 *              interpolation of S at the source wavelength lambda_m / (1 + f(beta))
 *   active     InfoMap P:208 (later region in list order overrides), Eq. 3 P:79 per covered cell,
 *              summed over covered cells; sign of BASELINE.json north_star: delta = active - quiet,
 *              so that S_final = S_quiet,integrated + delta (Eq. 4 P:83 with the sign flipped)
 *   mu bins    "closest mu" P:332
 *   contrast   per-pixel I_ratio applied after the shift, LB(mu) per cell
 *   effects    flux-only / CB-only differences, Eq. 1-2 P:73-77 (soap_oracle_active_effect)
 *   diff. rot. omega = omega_0 + omega_1 sin^2(latitude) P:250-252 (oracle_star.diff_rot = omega_1 / omega_0)
 *   resolution "lower the resolution of the final spectrum" P:85, Alg. 5: Gaussian LSF of FWHM lambda / R
 *              (reading R-LSF; soap_oracle_lower_resolution)
 *   line RV    first-moment RV per line, BASELINE.json north_star's acceptance functional standing in for
 *              the CCF fit of P:270 (soap_oracle_line_rvs)
 *   SOAPcontrast  "derives the contrast by calculating the ratio of two Planck functions at two different effective
 *              temperatures", one value per wavelength pixel, P:312 (and P:300 for SOAP 2.0's single-wavelength
 *              version of it) (soap_oracle_contrast_planck)
 *
 * No blocking, fusion or reordering: per output pixel the cells are summed in (j, i) order exactly
 * as the double loop of Alg. 1 would.  OpenMP only splits the *wavelength* axis into chunks, which
 * leaves every pixel's summation order untouched (results are bit-identical for any thread count).
 *
 * Shares no code, header, table or helper with the CUDA path (paper_2301_04259_b200/csrc).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.
 *
 * Parity status: pinned against closed forms / invariants / brute force (tests/test_oracle_pins.py,
 * pins P1-P10 of DESIGN.md; tests/test_oracle_effects.py, test_oracle_diffrot.py, test_oracle_lsf.py,
 * test_oracle_rv.py, test_oracle_contrast.py for the additions); "parity against values printed in the paper": unpinned - the paper
 * prints no numeric output for this path.
 *
 * Cell indexing everywhere: c = j * N + i, j = column (x) index, i = row (y) index,
 * x_j = -1 + (2 j + 1)/N, y_i = -1 + (2 i + 1)/N.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SOAP_C_KMS 299792.458
#define ORACLE_PI 3.14159265358979323846

typedef struct {
    int32_t grid_n;
    double vsini_kms, incl_deg, ld_u1, ld_u2;
    int32_t n_mu;
    const double *mu_centres; /* ascending */
    int32_t doppler_mode;     /* 0: relativistic (Eq. 6), 1: first order lambda (1 - v/c) */
    double diff_rot;          /* omega_1 / omega_0 of omega = omega_0 + omega_1 sin^2(theta); 0 = solid body */
} oracle_star;

typedef struct {
    double lat_deg, lon_deg, radius;
    int32_t type; /* 1 spot, 2 facula */
} oracle_region;

int soap_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void soap_oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* "closest mu"; exact tie -> larger mu; outside the centres -> end bin (reading S9). */
static int32_t nearest_bin(double mu, int32_t n_mu, const double *centres) {
    int32_t best = 0;
    double bd = fabs(mu - centres[0]);
    for (int32_t b = 1; b < n_mu; ++b) {
        double d = fabs(mu - centres[b]);
        if (d <= bd) { /* <= : on a tie the later (larger-mu) centre wins */
            bd = d;
            best = b;
        }
    }
    return best;
}

/* Doppler factor D: source wavelength = lambda_m * D.
 * mode 0: Eq. 6, lambda' = lambda (1 + f), 1 + f = sqrt((1+beta)/(1-beta))  =>  D = sqrt((1-beta)/(1+beta)).
 * mode 1: D = 1 - beta  (the lambda(1 - v/c) of BASELINE.json north_star). */
static double doppler_factor(double v_kms, int32_t mode) {
    double beta = v_kms / SOAP_C_KMS;
    if (mode == 1) return 1.0 - beta;
    return sqrt((1.0 - beta) / (1.0 + beta));
}

/*
 * Geometry (readings S1-S5, S9, S10).  All outputs are N*N arrays (any may be NULL).
 * Hidden cells (centre outside the unit disk) get visible = 0, mu = 0, w = 0, bin = -1, D = 1.
 * Returns the number of visible cells; *sum_w gets the sum of weights (visible cells, (j,i) order).
 */
int64_t soap_oracle_geometry(const oracle_star *st, double *x, double *y, double *mu, double *vel,
                             double *w, double *dfac, int32_t *bin, uint8_t *visible, double *sum_w) {
    const int32_t N = st->grid_n;
    const double sini = sin(st->incl_deg * ORACLE_PI / 180.0);
    const double cosi = cos(st->incl_deg * ORACLE_PI / 180.0);
    int64_t nvis = 0;
    double sw = 0.0;
    for (int32_t j = 0; j < N; ++j) {
        for (int32_t i = 0; i < N; ++i) {
            const int64_t c = (int64_t)j * N + i;
            const double xc = -1.0 + (2.0 * j + 1.0) / N;
            const double yc = -1.0 + (2.0 * i + 1.0) / N;
            const double r2 = xc * xc + yc * yc;
            const int vis = (r2 <= 1.0);
            double m = 0.0, ww = 0.0, v = 0.0, D = 1.0;
            int32_t b = -1;
            if (vis) {
                double a = 1.0 - r2;
                m = sqrt(a > 0.0 ? a : 0.0);
                v = xc * st->vsini_kms * sini;
                if (st->diff_rot != 0.0) {
                    /* differential rotation (reading R-DR): the surface point (x, y, mu) of the
                     * observer frame has sin(latitude) = y sin i + mu cos i (inverse of the tilt of reading S13) and
                     * rotates at omega_0 (1 + diff_rot sin^2 latitude); its line-of-sight velocity is x omega R sin i */
                    const double sinth = yc * sini + m * cosi;
                    v = v * (1.0 + st->diff_rot * sinth * sinth);
                }
                ww = 1.0 - st->ld_u1 * (1.0 - m) - st->ld_u2 * (1.0 - m) * (1.0 - m);
                b = nearest_bin(m, st->n_mu, st->mu_centres);
                D = doppler_factor(v, st->doppler_mode);
                nvis++;
                sw += ww;
            }
            if (x) x[c] = xc;
            if (y) y[c] = yc;
            if (mu) mu[c] = m;
            if (vel) vel[c] = v;
            if (w) w[c] = ww;
            if (dfac) dfac[c] = D;
            if (bin) bin[c] = b;
            if (visible) visible[c] = (uint8_t)vis;
        }
    }
    if (sum_w) *sum_w = sw;
    return nvis;
}

/*
 * The per-cell operation of Alg. 1 lines 3-4 / Eq. 5-9 as a gather: value at pixel m of the row S
 * Doppler-shifted by factor D and interpolated back onto the grid
 *   == numpy.interp(lam * D, lam, S)[m]   (clamped to the end values outside the grid, reading S8).
 */
static inline double shifted_at(const double *S, int64_t P, double lambda0, double k, double D, int64_t m) {
    const double lam_m = lambda0 + (double)m * k;
    const double src = lam_m * D;
    const double lam_last = lambda0 + (double)(P - 1) * k;
    if (src <= lambda0) return S[0];
    if (src >= lam_last) return S[P - 1];
    const double u = (src - lambda0) / k; /* Eq. 7-8: the bracketing index, closed form */
    int64_t n = (int64_t)floor(u);
    if (n > P - 2) n = P - 2;
    const double t = u - (double)n;
    return S[n] + t * (S[n + 1] - S[n]); /* Eq. 9 */
}

/* Exposed so that tests can pin the per-cell operation against numpy.interp (pin P8). */
void soap_oracle_shifted_row(const double *S, int64_t P, double lambda0, double k, double D,
                             int64_t m_lo, int64_t m_hi, double *out) {
    for (int64_t m = m_lo; m < m_hi; ++m) out[m - m_lo] = shifted_at(S, P, lambda0, k, D, m);
}

#define ORACLE_CHUNK 2048

/*
 * Alg. 1: Q[m] = sum over visible cells of w * shifted(S_quiet[bin], D)[m], for pixels
 * m_lo <= m < m_hi (the full spectrum is m_lo = 0, m_hi = P; a sub-range lets tests sample big configs).
 * S is [n_mu][P] row-major.  out has m_hi - m_lo entries.
 */
int soap_oracle_quiet(const oracle_star *st, const double *S, int64_t P, double lambda0, double k,
                      int64_t m_lo, int64_t m_hi, double *out) {
    const int32_t N = st->grid_n;
    const int64_t ncell = (int64_t)N * N;
    double *w = (double *)malloc(sizeof(double) * ncell);
    double *D = (double *)malloc(sizeof(double) * ncell);
    int32_t *bin = (int32_t *)malloc(sizeof(int32_t) * ncell);
    uint8_t *vis = (uint8_t *)malloc(ncell);
    if (!w || !D || !bin || !vis) return -1;
    soap_oracle_geometry(st, NULL, NULL, NULL, NULL, w, D, bin, vis, NULL);
    const int64_t n_out = m_hi - m_lo;
    const int64_t n_chunks = (n_out + ORACLE_CHUNK - 1) / ORACLE_CHUNK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        const int64_t a = m_lo + ch * ORACLE_CHUNK;
        const int64_t b = (a + ORACLE_CHUNK < m_hi) ? a + ORACLE_CHUNK : m_hi;
        for (int64_t m = a; m < b; ++m) out[m - m_lo] = 0.0;
        for (int32_t j = 0; j < N; ++j) {
            for (int32_t i = 0; i < N; ++i) {
                const int64_t c = (int64_t)j * N + i;
                if (!vis[c]) continue;
                const double *row = S + (int64_t)bin[c] * P;
                const double wc = w[c], Dc = D[c];
                for (int64_t m = a; m < b; ++m)
                    out[m - m_lo] += wc * shifted_at(row, P, lambda0, k, Dc, m);
            }
        }
    }
    free(w); free(D); free(bin); free(vis);
    return 0;
}

/*
 * InfoMap of Alg. 5 for one phase: type[c] = type of the LAST region in list order that
 * covers visible cell c, else 0.  Region centre (readings S11-S14):
 *   star frame   s = (cos lat sin L, sin lat, cos lat cos L),  L = lon + 2 pi phase
 *   observer     (xr, yr, zr) = (s_x, s_y sin i - s_z cos i, s_y cos i + s_z sin i)
 *   cell (x, y, mu) is covered  <=>  x xr + y yr + mu zr >= sqrt(1 - radius^2)
 * Returns the number of covered (active) cells.
 */
int64_t soap_oracle_info_map(const oracle_star *st, const oracle_region *regions, int32_t n_regions,
                             double phase, int32_t *type_map) {
    const int32_t N = st->grid_n;
    const double inc = st->incl_deg * ORACLE_PI / 180.0;
    const double si = sin(inc), ci = cos(inc);
    int64_t n_active = 0;
    for (int64_t c = 0; c < (int64_t)N * N; ++c) type_map[c] = 0;
    for (int32_t r = 0; r < n_regions; ++r) {
        const double lat = regions[r].lat_deg * ORACLE_PI / 180.0;
        const double L = regions[r].lon_deg * ORACLE_PI / 180.0 + 2.0 * ORACLE_PI * phase;
        const double sx = cos(lat) * sin(L), sy = sin(lat), sz = cos(lat) * cos(L);
        const double xr = sx, yr = sy * si - sz * ci, zr = sy * ci + sz * si;
        const double rad = regions[r].radius;
        const double cos_alpha = sqrt(1.0 - rad * rad);
        for (int32_t j = 0; j < N; ++j) {
            for (int32_t i = 0; i < N; ++i) {
                const double xc = -1.0 + (2.0 * j + 1.0) / N;
                const double yc = -1.0 + (2.0 * i + 1.0) / N;
                const double r2 = xc * xc + yc * yc;
                if (!(r2 <= 1.0)) continue;
                const double a = 1.0 - r2;
                const double m = sqrt(a > 0.0 ? a : 0.0);
                if (xc * xr + yc * yr + m * zr >= cos_alpha) type_map[(int64_t)j * N + i] = regions[r].type;
            }
        }
    }
    for (int64_t c = 0; c < (int64_t)N * N; ++c) n_active += (type_map[c] != 0);
    return n_active;
}

/*
 * Alg. 5 + Eq. 3, north_star sign:
 *   delta[p][m] = sum over cells with type t != 0 of
 *                 w * ( C_t[m] * LB_t(mu) * shifted(S_t[bin], D)[m] - shifted(S_quiet[bin], D)[m] )
 * S_quiet, S_spot, S_facula: [n_mu][P] (spot / facula may be NULL if no region of that type exists);
 * C_spot, C_facula: [P] or NULL (== 1);  lb_spot, lb_facula: 3 polynomial coefficients each.
 * delta: [n_phases][m_hi - m_lo];  n_active: [n_phases] or NULL.
 * Returns 0, or -2 if a region needs a spectrum that is NULL.
 */
int soap_oracle_active_effect(const oracle_star *st, const double *S_quiet, const double *S_spot,
                              const double *S_facula, const double *C_spot, const double *C_facula,
                              const double *lb_spot, const double *lb_facula, int64_t P, double lambda0,
                              double k, const oracle_region *regions, int32_t n_regions,
                              const double *phases, int32_t n_phases, int64_t m_lo, int64_t m_hi,
                              int32_t effect, double *delta, int32_t *n_active);

int soap_oracle_active(const oracle_star *st, const double *S_quiet, const double *S_spot,
                       const double *S_facula, const double *C_spot, const double *C_facula,
                       const double *lb_spot, const double *lb_facula, int64_t P, double lambda0,
                       double k, const oracle_region *regions, int32_t n_regions, const double *phases,
                       int32_t n_phases, int64_t m_lo, int64_t m_hi, double *delta, int32_t *n_active) {
    return soap_oracle_active_effect(st, S_quiet, S_spot, S_facula, C_spot, C_facula, lb_spot, lb_facula, P,
                                     lambda0, k, regions, n_regions, phases, n_phases, m_lo, m_hi, 0, delta,
                                     n_active);
}

/* The three effects of PAPER.md:73-79, per covered cell, with north_star's sign (active minus quiet: the
 * negatives of Eq. 1-3), I_ratio = C_t[m] * LB_t(mu_c):
 *   effect 0 (total, Eq. 3):      w * ( I_ratio * S'_active - S'_quiet )
 *   effect 1 (flux only, Eq. 1):  w * ( I_ratio * S'_quiet  - S'_quiet )
 *   effect 2 (CB only, Eq. 2):    w * (           S'_active - S'_quiet )
 * Everything else as soap_oracle_active.  Returns -4 for an unknown effect. */
int soap_oracle_active_effect(const oracle_star *st, const double *S_quiet, const double *S_spot,
                              const double *S_facula, const double *C_spot, const double *C_facula,
                              const double *lb_spot, const double *lb_facula, int64_t P, double lambda0,
                              double k, const oracle_region *regions, int32_t n_regions,
                              const double *phases, int32_t n_phases, int64_t m_lo, int64_t m_hi,
                              int32_t effect, double *delta, int32_t *n_active) {
    if (effect < 0 || effect > 2) return -4;
    const int32_t N = st->grid_n;
    const int64_t ncell = (int64_t)N * N;
    for (int32_t r = 0; r < n_regions; ++r) {
        if (regions[r].type == 1 && !S_spot) return -2;
        if (regions[r].type == 2 && !S_facula) return -2;
        if (regions[r].type != 1 && regions[r].type != 2) return -3;
    }
    double *w = (double *)malloc(sizeof(double) * ncell);
    double *mu = (double *)malloc(sizeof(double) * ncell);
    double *D = (double *)malloc(sizeof(double) * ncell);
    int32_t *bin = (int32_t *)malloc(sizeof(int32_t) * ncell);
    int32_t *type_map = (int32_t *)malloc(sizeof(int32_t) * ncell);
    if (!w || !mu || !D || !bin || !type_map) return -1;
    soap_oracle_geometry(st, NULL, NULL, mu, NULL, w, D, bin, NULL, NULL);
    const int64_t n_out = m_hi - m_lo;
    const int64_t n_chunks = (n_out + ORACLE_CHUNK - 1) / ORACLE_CHUNK;
    for (int32_t p = 0; p < n_phases; ++p) {
        int64_t na = soap_oracle_info_map(st, regions, n_regions, phases[p], type_map);
        if (n_active) n_active[p] = (int32_t)na;
        double *dp = delta + (int64_t)p * n_out;
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t ch = 0; ch < n_chunks; ++ch) {
            const int64_t a = m_lo + ch * ORACLE_CHUNK;
            const int64_t b = (a + ORACLE_CHUNK < m_hi) ? a + ORACLE_CHUNK : m_hi;
            for (int64_t m = a; m < b; ++m) dp[m - m_lo] = 0.0;
            if (na == 0) continue; /* reading S19: empty phase -> exact zeros */
            for (int32_t j = 0; j < N; ++j) {
                for (int32_t i = 0; i < N; ++i) {
                    const int64_t c = (int64_t)j * N + i;
                    const int32_t t = type_map[c];
                    if (t == 0) continue;
                    const double *rq = S_quiet + (int64_t)bin[c] * P;
                    const double *ra = (t == 1 ? S_spot : S_facula) + (int64_t)bin[c] * P;
                    const double *C = (t == 1 ? C_spot : C_facula);
                    const double *lbc = (t == 1 ? lb_spot : lb_facula);
                    const double lb = lbc[0] + lbc[1] * mu[c] + lbc[2] * mu[c] * mu[c];
                    const double wc = w[c], Dc = D[c];
                    for (int64_t m = a; m < b; ++m) {
                        const double cm = C ? C[m] : 1.0;
                        const double sq = shifted_at(rq, P, lambda0, k, Dc, m);
                        if (effect == 0)
                            dp[m - m_lo] += wc * (cm * lb * shifted_at(ra, P, lambda0, k, Dc, m) - sq);
                        else if (effect == 1)
                            dp[m - m_lo] += wc * (cm * lb * sq - sq);
                        else
                            dp[m - m_lo] += wc * (shifted_at(ra, P, lambda0, k, Dc, m) - sq);
                    }
                }
            }
        }
    }
    free(w); free(mu); free(D); free(bin); free(type_map);
    return 0;
}

/* Resolution lowering (Alg. 2, Alg. 5: "lower the resolution of the final spectrum to
 * match the resolution provided in the configuration file").  The paper names no kernel; reading R-LSF:
 * a Gaussian line-spread function of FWHM lambda / R, sampled on the pixel grid at every output pixel,
 *   sigma_m = lambda_m / (R * 2 sqrt(2 ln 2)),   g_m(j) = exp(-(j k)^2 / (2 sigma_m^2)),   |j| <= J_m = ceil(nsig sigma_m / k),
 *   out[m] = sum_j g_m(j) in[clamp(m + j, 0, P-1)] / sum_j g_m(j)
 * (discretely normalised, ends clamped like reading S8).  in / out: [n_rows][P], rows independent.  R <= 0 copies. */
int soap_oracle_lower_resolution(const double *in, int64_t n_rows, int64_t P, double lambda0, double k,
                                 double R, double nsig, double *out) {
    if (!in || !out || P < 1 || n_rows < 0 || !(k > 0.0) || !(nsig > 0.0)) return -1;
    const double fwhm_to_sigma = 1.0 / (2.0 * sqrt(2.0 * log(2.0)));
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < P; ++m) {
        if (!(R > 0.0)) {
            for (int64_t r = 0; r < n_rows; ++r) out[r * P + m] = in[r * P + m];
            continue;
        }
        const double lam = lambda0 + k * (double)m;
        const double sigma = lam / R * fwhm_to_sigma;
        const int64_t J = (int64_t)ceil(nsig * sigma / k);
        double norm = 0.0;
        for (int64_t j = -J; j <= J; ++j) {
            const double d = (double)j * k;
            norm += exp(-(d * d) / (2.0 * sigma * sigma));
        }
        for (int64_t r = 0; r < n_rows; ++r) {
            const double *row = in + r * P;
            double acc = 0.0;
            for (int64_t j = -J; j <= J; ++j) {
                int64_t n = m + j;
                if (n < 0) n = 0;
                if (n > P - 1) n = P - 1;
                const double d = (double)j * k;
                acc += exp(-(d * d) / (2.0 * sigma * sigma)) * row[n];
            }
            out[r * P + m] = acc / norm;
        }
    }
    return 0;
}

/* First-moment radial velocity of spectral lines: the acceptance functional of BASELINE.json north_star ("a
 * first-moment RV of each line"), made concrete in SURVEY section 8c; it stands in for the paper's CCF + Gaussian
 * fit, whose mask is not available.  For row r and line l with centre lc and window half-width hw:
 *   pixels m_lo = ceil((lc - hw - lambda0)/k) .. m_hi = floor((lc + hw - lambda0)/k)  (inclusive),
 *   f = F[r][m] / norm[r],  depth = 1 - f,
 *   rv[r][l] = c * sum_m (lambda_m - lc) depth / sum_m depth / lc          [cm/s, c = 299792.458e5]
 * NaN when the window is not inside [edge, P - edge) or the depth sum is 0.  rows: [n_rows][P]; rv: [n_rows][n_lines]. */
int soap_oracle_line_rvs(const double *rows, int64_t n_rows, int64_t P, double lambda0, double k,
                         const double *centres, const double *half_widths, int64_t n_lines, const double *norm,
                         int64_t edge, double *rv) {
    if (!rows || !centres || !half_widths || !norm || !rv || P < 1 || !(k > 0.0)) return -1;
    const double c_cms = SOAP_C_KMS * 1e5;
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < n_lines; ++l) {
        const double lc = centres[l], hw = half_widths[l];
        const int64_t m_lo = (int64_t)ceil((lc - hw - lambda0) / k);
        const int64_t m_hi = (int64_t)floor((lc + hw - lambda0) / k);
        const int ok = (m_lo >= edge) && (m_hi < P - edge) && (m_hi >= m_lo);
        for (int64_t r = 0; r < n_rows; ++r) {
            double num = 0.0, den = 0.0;
            if (ok) {
                for (int64_t m = m_lo; m <= m_hi; ++m) {
                    const double depth = 1.0 - rows[r * P + m] / norm[r];
                    num += ((lambda0 + k * (double)m) - lc) * depth;
                    den += depth;
                }
            }
            rv[r * n_lines + l] = (ok && den != 0.0) ? c_cms * num / den / lc : NAN;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * SOAPcontrast: "each wavelength pixel is first accessed by the global index of the kernel.  Next on each
 * thread, it derives the contrast by calculating the ratio of two Planck functions at two different effective
 * temperatures."  With B_lambda(T) = (2 h c^2 / lambda^5) / (exp(h c / (lambda k_B T)) - 1) the prefactor cancels:
 *     contrast[m] = B_lambda_m(T_active) / B_lambda_m(T_quiet) = (exp(x_q) - 1) / (exp(x_a) - 1),  x = h c / (lambda_m k_B T),
 * lambda_m = lambda0 + m k in Angstrom (the unit of every wavelength in BASELINE.json's configs).  This is the
 * I_ratio of Eq. 3 that multiplies the shifted active spectrum.  Constants: CODATA 2018 exact values.
 * ------------------------------------------------------------------------------------------------ */
#define ORACLE_PLANCK_H 6.62607015e-34 /* J s */
#define ORACLE_BOLTZMANN 1.380649e-23  /* J / K */
#define ORACLE_C_MS 299792458.0        /* m / s */

int soap_oracle_contrast_planck(double lambda0, double k, int64_t n_pix, double T_quiet, double T_active, double *out) {
    if (!(T_quiet > 0.0) || !(T_active > 0.0) || !(lambda0 > 0.0) || !(k > 0.0) || n_pix < 0) return -1;
    const double hc_over_kb = ORACLE_PLANCK_H * ORACLE_C_MS / ORACLE_BOLTZMANN; /* m K */
    for (int64_t m = 0; m < n_pix; ++m) {
        const double lam_m = (lambda0 + k * (double)m) * 1e-10; /* Angstrom -> metre */
        const double xq = hc_over_kb / (lam_m * T_quiet), xa = hc_over_kb / (lam_m * T_active);
        out[m] = expm1(xq) / expm1(xa);
    }
    return 0;
}
