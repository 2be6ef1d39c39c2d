// First-moment radial velocity of spectral lines on the device ("then a CCF / first-moment RV
// reduction on device"): the acceptance functional of BASELINE.json north_star, standing in for the paper's CCF + Gaussian
// fit, whose mask is not available.  For row r and line l (centre lc, window half-width hw):
//   m_lo = ceil((lc - hw - lambda0)/k) .. m_hi = floor((lc + hw - lambda0)/k),  depth = 1 - F[r][m] / norm[r],
//   rv[r][l] = c sum_m (lambda_m - lc) depth / sum_m depth / lc  [cm/s];  NaN if the window leaves [edge, P - edge) or depth sums to 0.
// One warp per line, one lane per row: fp64 sums in ascending pixel order (deterministic).
// HBM-bound: every row is read about once (windows of neighbouring lines overlap in L2).
#pragma once
#include <cmath>
#include <cstdint>
#include <cuda_runtime.h>

namespace soap {

constexpr int kRvWarps = 8;

struct RvArgs {
    const void *rows;
    long long n_rows, n_pix, pitch;
    double lambda0, k;
    const double *centres, *half_widths;  // DEVICE [n_lines]
    const double *norm;                   // DEVICE [n_rows]
    long long n_lines, edge;
    double *rv;                           // DEVICE [n_rows][n_lines]
};

template <typename T>
__global__ void __launch_bounds__(32 * kRvWarps) line_rv_kernel(const RvArgs a) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long l = (long long)blockIdx.x * kRvWarps + warp;
    if (l >= a.n_lines) return;
    const double lc = a.centres[l], hw = a.half_widths[l];
    const long long m_lo = (long long)ceil(__ddiv_rn(__dadd_rn(__dadd_rn(lc, -hw), -a.lambda0), a.k));
    const long long m_hi = (long long)floor(__ddiv_rn(__dadd_rn(__dadd_rn(lc, hw), -a.lambda0), a.k));
    const bool ok = m_lo >= a.edge && m_hi < a.n_pix - a.edge && m_hi >= m_lo;
    const T *rows = static_cast<const T *>(a.rows);
    const double c_cms = 299792.458e5;
    // lane = row: the (line-dependent) window arithmetic above is done once per warp, every lane then walks the ~20-50
    // pixels of its own row's window in ascending order (the order of the definition); the rows' sectors are reused
    // from L1 across the iterations
    for (long long r = (long long)blockIdx.y * 32 + lane; r < a.n_rows; r += 32LL * gridDim.y) {
        double num = 0.0, den = 0.0;
        if (ok) {
            const T *row = rows + r * a.pitch;
            const double inv_norm = 1.0 / a.norm[r];  // one division per (line, row): 1 ulp from the per-pixel quotient
            for (long long m = m_lo; m <= m_hi; ++m) {
                const double depth = 1.0 - (double)row[m] * inv_norm;
                num += (__dadd_rn(a.lambda0, __dmul_rn(a.k, (double)m)) - lc) * depth;
                den += depth;
            }
        }
        a.rv[r * a.n_lines + l] = (ok && den != 0.0) ? c_cms * num / den / lc : nan("");
    }
}

}  // namespace soap
