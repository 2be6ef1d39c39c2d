// First-moment radial velocity of spectral lines on the device ("then a CCF / first-moment RV
// reduction on device"): the acceptance functional of BASELINE.json north_star, standing in for the paper's CCF + Gaussian
// fit, whose mask is not available.  For row r and line l (centre lc, window half-width hw):
//   m_lo = ceil((lc - hw - lambda0)/k) .. m_hi = floor((lc + hw - lambda0)/k),  depth = 1 - F[r][m] / norm[r],
//   rv[r][l] = c sum_m (lambda_m - lc) depth / sum_m depth / lc  [cm/s];  NaN if the window leaves [edge, P - edge) or depth sums to 0.
// One warp per line.  The line's window of every row is first brought into shared memory with asynchronous copies - lanes
// over consecutive pixels of one row: coalesced, every copy of the window in flight at once - and then summed with one
// lane per row in ascending pixel order (the order of the definition; fp64, deterministic) from a row-major tile whose
// odd pitch keeps the lanes on distinct banks.  (One lane per row reading global memory directly costs one L1 wavefront
// per row and pixel: 25x the traffic through the L1 tag stage, and that stage - not HBM - bound the kernel.)
// HBM-bound: every row is read about once (windows of neighbouring lines overlap in L2).
#pragma once
#include <cmath>
#include <cstdint>
#include <cuda_runtime.h>

#include "ptx_helpers.cuh"

namespace soap {

constexpr int kRvWarps = 8;
constexpr int kRvRows = 32;  // rows per pass at most: one lane each

struct RvArgs {
    const void *rows;
    long long n_rows, n_pix, pitch;
    double lambda0, k;
    const double *centres, *half_widths;  // DEVICE [n_lines]
    const double *norm;                   // DEVICE [n_rows]
    long long n_lines, edge;
    double *rv;                           // DEVICE [n_rows][n_lines]
    int rows_pass;                        // rows staged per pass: min(kRvRows, n_rows) - sizes the shared-memory tiles
};

template <typename T>
__host__ __device__ constexpr int rv_chunk() { return sizeof(T) == 4 ? 48 : 32; }  // window pixels staged per pass (most
                                                                                   // windows fit in one; wider ones take several)
template <typename T>
__host__ __device__ constexpr size_t rv_warp_bytes(int rows_pass) {  // per warp: the row-major tile, then lambda_m - lc of its pixels (fp64)
    return (((size_t)rows_pass * (rv_chunk<T>() + 1) * sizeof(T) + 7) & ~(size_t)7) + (size_t)rv_chunk<T>() * sizeof(double);
}
template <typename T>
__host__ __device__ constexpr size_t rv_smem_bytes(int rows_pass) { return (size_t)kRvWarps * rv_warp_bytes<T>(rows_pass); }

template <typename T>
__global__ void __launch_bounds__(32 * kRvWarps) line_rv_kernel(const RvArgs a) {
    extern __shared__ __align__(16) unsigned char rv_smem[];
    constexpr int CH = rv_chunk<T>(), PITCH = CH + 1;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const size_t wbytes = rv_warp_bytes<T>(a.rows_pass);
    T *tile = reinterpret_cast<T *>(rv_smem + (size_t)warp * wbytes);  // [rows_pass][PITCH]
    double *dl = reinterpret_cast<double *>(rv_smem + (size_t)(warp + 1) * wbytes) - CH;  // [CH]
    const long long l = (long long)blockIdx.x * kRvWarps + warp;
    if (l >= a.n_lines) return;
    const double lc = a.centres[l], hw = a.half_widths[l];
    const long long m_lo = (long long)ceil(__ddiv_rn(__dadd_rn(__dadd_rn(lc, -hw), -a.lambda0), a.k));
    const long long m_hi = (long long)floor(__ddiv_rn(__dadd_rn(__dadd_rn(lc, hw), -a.lambda0), a.k));
    const bool ok = m_lo >= a.edge && m_hi < a.n_pix - a.edge && m_hi >= m_lo;
    const T *rows = static_cast<const T *>(a.rows);
    const double c_cms = 299792.458e5;
    for (long long r0 = (long long)blockIdx.y * a.rows_pass; r0 < a.n_rows; r0 += (long long)a.rows_pass * gridDim.y) {
        const int nr = (int)min((long long)a.rows_pass, a.n_rows - r0);
        const long long r = r0 + lane;
        const bool mine = lane < nr;
        double num = 0.0, den = 0.0;
        if (ok) {
            const double inv_norm = mine ? 1.0 / a.norm[r] : 0.0;  // one division per (line, row): 1 ulp from the per-pixel quotient
            for (long long c0 = m_lo; c0 <= m_hi; c0 += CH) {
                const int cw = (int)min((long long)CH, m_hi - c0 + 1);
                {  // lane i copies pixels i (and i + 32) of every row: pointers advance by one row per step
                    const T *src = rows + r0 * a.pitch + c0 + lane;
                    T *dst = tile + lane;
                    const bool p0 = lane < cw, p1 = CH > 32 && lane + 32 < cw;
#pragma unroll 4
                    for (int rr = 0; rr < nr; ++rr, src += a.pitch, dst += PITCH) {
                        if (sizeof(T) == 4) {
                            if (p0) cp_async_4(dst, src);
                            if (p1) cp_async_4(dst + 32, src + 32);
                        } else {
                            if (p0) cp_async_8(dst, src);
                        }
                    }
                }
                cp_async_commit();
                // lambda_m - lc depends on the pixel only: once per pixel (lanes over pixels), not once per row and pixel
                for (int i = lane; i < cw; i += 32) dl[i] = __dadd_rn(a.lambda0, __dmul_rn(a.k, (double)(c0 + i))) - lc;
                cp_async_wait_all();
                __syncwarp();
                if (mine) {
                    const T *mr = tile + lane * PITCH;
#pragma unroll 4
                    for (int i = 0; i < cw; ++i) {
                        const double depth = fma(-(double)mr[i], inv_norm, 1.0);
                        num += dl[i] * depth;
                        den += depth;
                    }
                }
                __syncwarp();
            }
        }
        if (mine) a.rv[r * a.n_lines + l] = (ok && den != 0.0) ? c_cms * num / den / lc : nan("");
    }
}

}  // namespace soap
