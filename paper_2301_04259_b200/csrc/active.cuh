// a4 of SURVEY section 8: per-phase active map and compaction (InfoMap of Alg. 5).
//
// The paper rewrites an N x N type map on the device at every timestamp.  Here the map is never
// materialised: one thread per (phase, column) walks its column, decides each cell's type by spherical
// angular distance with list-order override, and bins the covered cells by (mu-bin, kind) - all cells
// of a column share one velocity - and a second kernel compacts the non-zero bins of every
// (phase, kind, mu-bin) into the entry list the shift-interpolate-accumulate kernel consumes.
// Kinds: 0 = quiet row of a covered cell (weight -w), 1 = spot row, 2 = facula row (weight +w LB_t(mu)).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "geometry.cuh"

namespace soap {

struct RegionAtPhase {  // region centre in the observer frame at one phase (host-computed, fp64)
    double xr, yr, zr;
    double cos_alpha;   // sqrt(1 - radius^2): covered <=> x xr + y yr + mu zr >= cos_alpha
    double chord;       // 2 sin(alpha/2): max distance between a covered surface point and the centre
    int type;           // 1 spot, 2 facula; 0 = skip (entirely on the far side)
    int pad;
};

struct LbCoef {
    double c[3][3];  // [kind][power]; kind 0 unused
};

constexpr int kBinWarps = 8;  // warps (columns) per CTA of active_bin_kernel

// grid: (ceil(N/kBinWarps), n_phases); one warp per (phase, column), lanes over the rows (coalesced).
// WD: [n_phases][3][n_mu][ncap] fp64, pre-zeroed.  Cells of equal (mu-bin, type) are contiguous in a
// column: segmented warp scans, added to WD in row order by one lane at a time (deterministic).
__global__ void __launch_bounds__(32 * kBinWarps)
active_bin_kernel(int N, int n_regions, int n_mu, int ncap, const RegionAtPhase *__restrict__ rp /*[n_phases][n_regions]*/,
                  const double *__restrict__ mu, const double *__restrict__ w, const int *__restrict__ bin, LbCoef lb,
                  double *__restrict__ WD, int *__restrict__ n_active /*[n_phases]*/) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int j = blockIdx.x * kBinWarps + warp;
    const int p = blockIdx.y;
    if (j >= N) return;
    const RegionAtPhase *reg = rp + (size_t)p * n_regions;
    const double x = cell_coord(j, N);
    // rows of this column that any region can reach (conservative: chord bound, slightly inflated)
    double ylo = 2.0, yhi = -2.0;
    for (int r = 0; r < n_regions; ++r) {
        if (reg[r].type == 0) continue;
        const double ch = reg[r].chord * (1.0 + 1e-9) + 1e-12;
        if (fabs(x - reg[r].xr) > ch) continue;
        ylo = fmin(ylo, reg[r].yr - ch);
        yhi = fmax(yhi, reg[r].yr + ch);
    }
    if (ylo > yhi) return;
    int i_lo = (int)floor((ylo + 1.0) * 0.5 * N - 0.5) - 1;
    int i_hi = (int)ceil((yhi + 1.0) * 0.5 * N - 0.5) + 1;
    i_lo = max(i_lo, 0);
    i_hi = min(i_hi, N - 1);
    double *WDp = WD + (size_t)p * 3 * n_mu * ncap;
    int count = 0;
    for (int i0 = i_lo; i0 <= i_hi; i0 += 32) {
        const int i = i0 + lane;
        int b = -1, t = 0;
        double wc = 0.0, wl = 0.0;
        if (i <= i_hi) {
            const size_t c = (size_t)j * N + i;
            b = bin[c];
            if (b >= 0) {
                const double y = cell_coord(i, N), m = mu[c];
                for (int r = 0; r < n_regions; ++r) {  // list order: the last covering region wins
                    if (reg[r].type == 0) continue;
                    const double dot =
                        __dadd_rn(__dadd_rn(__dmul_rn(x, reg[r].xr), __dmul_rn(y, reg[r].yr)), __dmul_rn(m, reg[r].zr));
                    if (dot >= reg[r].cos_alpha) t = reg[r].type;
                }
                if (t != 0) {
                    wc = w[c];
                    wl = wc * (lb.c[t][0] + lb.c[t][1] * m + lb.c[t][2] * m * m);
                }
            }
        }
        const int key = (t != 0) ? (b * 4 + t) : -1;
        int start;
        bool tail;
        const double seg_w = warp_segmented_scan(wc, key, lane, start, tail);
        const double seg_wl = warp_segmented_scan(wl, key, lane, start, tail);
        unsigned tails = __ballot_sync(0xffffffffu, tail && t != 0);
        while (tails) {
            const int l = __ffs(tails) - 1;
            if (lane == l) {
                WDp[((size_t)0 * n_mu + b) * ncap + j] += seg_w;
                WDp[((size_t)t * n_mu + b) * ncap + j] += seg_wl;
            }
            __syncwarp();
            tails &= tails - 1;
        }
        count += __popc(__ballot_sync(0xffffffffu, t != 0));
    }
    if (lane == 0 && count) atomicAdd(&n_active[p], count);  // integer: order-independent
}

// One warp per (phase, kind, mu-bin) segment: ordered compaction of the non-zero columns into
// entries (a_j, +-W).  Segment s = (p*3 + kind)*n_mu + b owns ent[s*ncap .. s*ncap + ncap); counts are
// padded to even with a zero-weight entry.  EntT = float2 or double2.
template <typename EntT>
__global__ void active_compact_kernel(int N, int n_mu, int ncap, int n_segments,
                                      const double *__restrict__ col_a, const double *__restrict__ WD,
                                      EntT *__restrict__ ent, int *__restrict__ seg_count,
                                      unsigned long long *__restrict__ total_entries) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= n_segments) return;
    const int kind = (warp / n_mu) % 3;
    const double sign = (kind == 0) ? -1.0 : 1.0;
    const double *src = WD + (size_t)warp * ncap;
    EntT *dst = ent + (size_t)warp * ncap;
    int pos = 0;
    for (int j0 = 0; j0 < N; j0 += 32) {
        const int j = j0 + lane;
        const double W = (j < N) ? src[j] : 0.0;
        const unsigned m = __ballot_sync(0xffffffffu, W != 0.0);
        if (W != 0.0) {
            EntT e;
            e.x = (decltype(e.x))col_a[j];
            e.y = (decltype(e.y))(sign * W);
            dst[pos + __popc(m & ((1u << lane) - 1u))] = e;
        }
        pos += __popc(m);
    }
    if (lane == 0) {
        if (pos & 1) {
            EntT z;
            z.x = 0;
            z.y = 0;
            dst[pos] = z;
        }
        seg_count[warp] = pos;
        if (pos) atomicAdd(total_entries, (unsigned long long)pos);
    }
}

}  // namespace soap
