// a1 + a2 of SURVEY section 8: disk geometry (Fig. 1) and (column, mu-bin) weight binning.
//
// All geometry is fp64 with explicitly rounded operations (no FMA contraction), so that the integer
// decisions taken here (visible / hidden, mu bin) are taken in the same precision as the fp64 definition.
// N^2 <= a few 10^5 cells: these kernels are launch-latency sized, not a cost centre.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "composite.cuh"
#include "ptx_helpers.cuh"

namespace soap {

constexpr double kSpeedOfLightKms = 299792.458;

struct DevInfo {            // device-resident summary, mirrored to soap_geom_info on request
    long long n_visible;
    long long n_entries;
    double sum_weights;
    double max_abs_dshift;
};

__device__ __forceinline__ double cell_coord(int idx, int N) {
    // -1 + (2 idx + 1)/N, each operation rounded once (reading S1)
    return __dadd_rn(-1.0, __ddiv_rn(__dadd_rn(__dmul_rn(2.0, (double)idx), 1.0), (double)N));
}

// One cell c = j*N + i: mu, limb-darkening weight, velocity and nearest mu bin (hidden: 0, 0, 0, -1).
struct Rotation {  // v_cell = x vsini sin i (1 + diff_rot sin^2 latitude)  (S5, reading R-DR)
    double vsini, sini, cosi, diff_rot;
};

__device__ __forceinline__ void cell_geometry(int j, int i, int N, const Rotation &rot, double u1, double u2, int n_mu,
                                              const double *__restrict__ mu_centres, double &mu, double &w, double &v,
                                              int &bin) {
    const double x = cell_coord(j, N), y = cell_coord(i, N);
    const double r2 = __dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y));
    mu = 0.0;
    w = 0.0;
    v = 0.0;
    bin = -1;
    if (r2 <= 1.0) {  // cell counts iff its centre is on the disk (reading S2)
        const double a = __dadd_rn(1.0, -r2);
        mu = __dsqrt_rn(a > 0.0 ? a : 0.0);
        v = __dmul_rn(__dmul_rn(x, rot.vsini), rot.sini);
        if (rot.diff_rot != 0.0) {  // sin(latitude) of the surface point (x, y, mu): inverse of the tilt of reading S13
            const double sinth = __dadd_rn(__dmul_rn(y, rot.sini), __dmul_rn(mu, rot.cosi));
            v = __dmul_rn(v, __dadd_rn(1.0, __dmul_rn(__dmul_rn(rot.diff_rot, sinth), sinth)));
        }
        const double om = __dadd_rn(1.0, -mu);
        // w = 1 - u1 (1-mu) - u2 (1-mu)^2, evaluated left to right
        w = __dadd_rn(__dadd_rn(1.0, -__dmul_rn(u1, om)), -__dmul_rn(__dmul_rn(u2, om), om));
        // closest mu centre; on an exact tie the larger mu wins (reading S9)
        double best = fabs(__dadd_rn(mu, -mu_centres[0]));
        bin = 0;
        for (int b = 1; b < n_mu; ++b) {
            const double d = fabs(__dadd_rn(mu, -mu_centres[b]));
            if (d <= best) {
                best = d;
                bin = b;
            }
        }
    }
}

// D - 1 without cancellation.  mode 0: D = sqrt((1-b)/(1+b))  =>  D - 1 = -2b / ((1+b) + sqrt(1-b^2));
// mode 1: D = 1 - b.
__device__ __forceinline__ double doppler_minus_one(double v_kms, int mode) {
    const double b = v_kms / kSpeedOfLightKms;
    if (mode == 1) return -b;
    return -2.0 * b / ((1.0 + b) + sqrt(1.0 - b * b));
}

// Inclusive segmented scan over the lanes of a warp: lanes with equal consecutive `key` form a segment;
// returns the sum of v over the lanes of the caller's segment up to and including the caller.  Fixed
// shuffle tree: deterministic.  `start` receives the first lane of the caller's segment.
__device__ __forceinline__ double warp_segmented_scan(double v, int key, int lane, int &start, bool &is_tail) {
    const int prev = __shfl_up_sync(0xffffffffu, key, 1);
    const bool head = (lane == 0) || (key != prev);
    const unsigned heads = __ballot_sync(0xffffffffu, head);
    start = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));
    is_tail = (lane == 31) || ((heads >> (lane + 1)) & 1u);
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane - d >= start) v += t;
    }
    return v;
}

constexpr int kGeomWarps = 32;  // warps (columns) per CTA of geometry_kernel

struct MuCentres {  // passed by value as a kernel argument: no host -> device copy per call
    double v[64];
};



// One warp, one column j, the 32-row chunks `chunk`, `chunk + stride`, ...: writes the cells' (mu, w, v, bin)
// and adds the chunk's binned weights to s_W[64] and cell counts to s_C[64] (segmented warp scans, in row order), returning
// the warp's weight sum and visible-cell count.
__device__ __forceinline__ void geometry_chunks(int j, int chunk, int stride, int N, const Rotation &rot, double u1, double u2,
                                                int n_mu, const double *s_mu, double *s_W, int *s_C, double *__restrict__ mu_out,
                                                double *__restrict__ w_out, double *__restrict__ vel_out,
                                                int *__restrict__ bin_out, double &sum, int &nvis) {
    const int lane = threadIdx.x & 31;
    sum = 0.0;
    nvis = 0;
    for (int i0 = 32 * chunk; i0 < N; i0 += 32 * stride) {
        const int i = i0 + lane;
        double mu = 0.0, w = 0.0, v = 0.0;
        int bin = -1;
        if (i < N) {
            cell_geometry(j, i, N, rot, u1, u2, n_mu, s_mu, mu, w, v, bin);
            const size_t c = (size_t)j * N + i;
            mu_out[c] = mu;
            w_out[c] = w;
            vel_out[c] = v;
            bin_out[c] = bin;
        }
        int start;
        bool tail;
        const double seg = warp_segmented_scan(w, bin, lane, start, tail);
        unsigned tails = __ballot_sync(0xffffffffu, tail && bin >= 0);
        while (tails) {  // segments of one bin may repeat inside a chunk (apex of the column): add in lane order
            const int l = __ffs(tails) - 1;
            if (lane == l) {
                s_W[bin] += seg;
                s_C[bin] += lane - start + 1;  // cells of the segment
            }
            __syncwarp();
            tails &= tails - 1;
        }
        double cs = w;  // chunk total, fixed xor tree
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) cs += __shfl_xor_sync(0xffffffffu, cs, d);
        sum += cs;
        nvis += __popc(__ballot_sync(0xffffffffu, bin >= 0));
    }
}

// Single CTA: compacts the non-zero W[j][b] into the entry list of the pre-binned form, sorted by
// (row b, column j), each row padded with a zero-weight entry to an even length so that every row
// starts 16-byte aligned for the TMA bulk copy; writes row_start[n_mu+1] and the summary.
// Entries are (a_j, W) in fp32 (float2) and fp64 (double2).
__device__ void build_binned_entries(int N, int n_mu, const double *col_a, const double *Wbin, const double *col_sumw,
                                     const int *col_nvis, float2 *ent32, double2 *ent64, int *row_start, DevInfo *info) {
    __shared__ int s_cnt[64];
    __shared__ int s_start[65];
    __shared__ long long s_nv[32];  // per-warp partial sums of the summary
    __shared__ double s_sw[32], s_am[32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
    constexpr int kBatch = 8;  // loads of 8 x 32 columns are issued together: one memory round trip per batch
    for (int b = warp; b < n_mu; b += n_warps) {
        int cnt = 0;
        for (int j0 = 0; j0 < N; j0 += 32 * kBatch) {
            double W[kBatch];
#pragma unroll
            for (int k = 0; k < kBatch; ++k) {
                const int j = j0 + 32 * k + lane;
                W[k] = (j < N) ? Wbin[(size_t)j * n_mu + b] : 0.0;
            }
#pragma unroll
            for (int k = 0; k < kBatch; ++k) cnt += __popc(__ballot_sync(0xffffffffu, W[k] != 0.0));
        }
        if (lane == 0) s_cnt[b] = cnt;
    }
    __syncthreads();
    // summary: per-thread strided partials, a fixed xor tree inside the warps, then the warps in order (deterministic)
    {
        long long nv = 0;
        double sw = 0.0, am = 0.0;
        for (int j = threadIdx.x; j < N; j += blockDim.x) {
            const int c = col_nvis[j];
            nv += c;
            sw += col_sumw[j];
            if (c > 0) am = fmax(am, fabs(col_a[j]));
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            nv += __shfl_xor_sync(0xffffffffu, nv, d);
            sw += __shfl_xor_sync(0xffffffffu, sw, d);
            am = fmax(am, __shfl_xor_sync(0xffffffffu, am, d));
        }
        if (lane == 0) {
            s_nv[warp] = nv;
            s_sw[warp] = sw;
            s_am[warp] = am;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < n_warps; ++w) {
            s_nv[0] += s_nv[w];
            s_sw[0] += s_sw[w];
            s_am[0] = fmax(s_am[0], s_am[w]);
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int off = 0, total = 0;
        for (int b = 0; b < n_mu; ++b) {
            s_start[b] = off;
            total += s_cnt[b];
            off += (s_cnt[b] + 1) & ~1;
        }
        s_start[n_mu] = off;
        info->n_visible = s_nv[0];
        info->n_entries = total;
        info->sum_weights = s_sw[0];
        info->max_abs_dshift = s_am[0];
    }
    __syncthreads();
    for (int b = threadIdx.x; b <= n_mu; b += blockDim.x) row_start[b] = s_start[b];
    for (int b = warp; b < n_mu; b += n_warps) {
        int pos = s_start[b];
        for (int j0 = 0; j0 < N; j0 += 32 * kBatch) {
            double W[kBatch], A[kBatch];
#pragma unroll
            for (int k = 0; k < kBatch; ++k) {
                const int j = j0 + 32 * k + lane;
                W[k] = (j < N) ? Wbin[(size_t)j * n_mu + b] : 0.0;
                A[k] = (j < N) ? col_a[j] : 0.0;
            }
#pragma unroll
            for (int k = 0; k < kBatch; ++k) {
                const unsigned m = __ballot_sync(0xffffffffu, W[k] != 0.0);
                if (W[k] != 0.0) {
                    const int e = pos + __popc(m & ((1u << lane) - 1u));
                    ent32[e] = make_float2((float)A[k], (float)W[k]);
                    ent64[e] = make_double2(A[k], W[k]);
                }
                pos += __popc(m);
            }
        }
        if (lane == 0 && (s_cnt[b] & 1)) {
            ent32[pos] = make_float2(0.f, 0.f);
            ent64[pos] = make_double2(0.0, 0.0);
        }
    }
}

// The same compaction - and the pair tables of the composite-column form (composite.cuh) - for grids whose binned
// weights fit in shared memory (fin_smem_bytes(N, n_mu) <= kFinSmemMax: every configuration of BASELINE.json).  The last
// CTA is alone on the critical path of the launch, and what it costs is dependent round trips to L2, not arithmetic:
// here W[j][b], a_j and the per-column sums are fetched ONCE, all loads in flight together, into a transposed
// shared-memory copy sW[b][j] (row pitch = 1 mod 16 doubles: conflict-free for the bin-major stores and the
// column-major reads); counts, prefix sums, entries and pair tables are then built from shared memory.
constexpr size_t kFinSmemMax = 160 * 1024;
__host__ __device__ inline int fin_pitch(int N) { return ((N + 14) / 16) * 16 + 1; }  // >= N, = 1 (mod 16)
__host__ __device__ inline size_t fin_smem_bytes(int N, int n_mu) {
    return ((size_t)n_mu * fin_pitch(N) + (size_t)N) * sizeof(double) + ((size_t)(N + 1) / 2 + 2) * sizeof(int);
}

__device__ void finalize_columns_smem(int N, int n_mu, const double *col_a, const double *Wbin, const double *col_sumw,
                                      const int *col_nvis, float2 *ent32, double2 *ent64, int *row_start, DevInfo *info,
                                      float2 *comp_Wp, int comp_stride, comp::PairHdr *comp_hdr, unsigned char *dyn) {
    __shared__ int s_cnt[64];
    __shared__ int s_start[65];
    __shared__ long long s_nv[32];
    __shared__ double s_sw[32], s_am[32];
    __shared__ int s_carry[33];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, n_warps = blockDim.x >> 5, nt = blockDim.x;
    const int Np = fin_pitch(N);
    double *sW = reinterpret_cast<double *>(dyn);  // [n_mu][Np]
    double *sA = sW + (size_t)n_mu * Np;           // [N]
    int *s_cost = reinterpret_cast<int *>(sA + N);  // [n_pairs + 1] exclusive cost prefix of the column pairs
    // ---- one round trip: every load is independent of every other (written by other SMs: read through L2) ----------
    // a warp takes a column at a time, lanes over the mu bins (no index arithmetic per element); four columns in flight
    long long nv = 0;
    double sw = 0.0, am = 0.0;
    constexpr int kInFlight = 4;
    for (int j0 = warp * kInFlight; j0 < N; j0 += n_warps * kInFlight) {
        for (int b0 = 0; b0 < n_mu; b0 += 32) {
            const int b = b0 + lane;
            double v[kInFlight];
#pragma unroll
            for (int u = 0; u < kInFlight; ++u) v[u] = (b < n_mu && j0 + u < N) ? __ldcg(&Wbin[(size_t)(j0 + u) * n_mu + b]) : 0.0;
#pragma unroll
            for (int u = 0; u < kInFlight; ++u)
                if (b < n_mu && j0 + u < N) sW[(size_t)b * Np + j0 + u] = v[u];
        }
    }
    for (int j = tid; j < N; j += nt) {
        const int c = __ldcg(&col_nvis[j]);
        const double a = __ldcg(&col_a[j]);
        sA[j] = a;
        nv += c;
        sw += __ldcg(&col_sumw[j]);
        if (c > 0) am = fmax(am, fabs(a));
    }
    // summary: fixed xor tree inside the warps, then over the warps (deterministic)
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        nv += __shfl_xor_sync(0xffffffffu, nv, d);
        sw += __shfl_xor_sync(0xffffffffu, sw, d);
        am = fmax(am, __shfl_xor_sync(0xffffffffu, am, d));
    }
    if (lane == 0) {
        s_nv[warp] = nv;
        s_sw[warp] = sw;
        s_am[warp] = am;
    }
    __syncthreads();  // sW, sA complete
    // ---- entries per mu bin ------------------------------------------------------------------------------------------
    for (int b = warp; b < n_mu; b += n_warps) {
        const double *row = sW + (size_t)b * Np;
        int cnt = 0;
        for (int j0 = 0; j0 < N; j0 += 32) {
            const int j = j0 + lane;
            cnt += __popc(__ballot_sync(0xffffffffu, j < N && row[j] != 0.0));
        }
        if (lane == 0) s_cnt[b] = cnt;
    }
    __syncthreads();
    if (warp == 0) {
        // row starts (rows padded to an even length) by a warp scan over <= 64 bins; the summary's last step
        int v0 = lane < n_mu ? ((s_cnt[lane] + 1) & ~1) : 0, v1 = lane + 32 < n_mu ? ((s_cnt[lane + 32] + 1) & ~1) : 0;
        int t0 = lane < n_mu ? s_cnt[lane] : 0, t1 = lane + 32 < n_mu ? s_cnt[lane + 32] : 0;
        int i0 = v0, i1 = v1;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int u0 = __shfl_up_sync(0xffffffffu, i0, d), u1 = __shfl_up_sync(0xffffffffu, i1, d);
            if (lane >= d) {
                i0 += u0;
                i1 += u1;
            }
        }
        const int first = __shfl_sync(0xffffffffu, i0, 31);
        s_start[lane] = i0 - v0;
        s_start[lane + 32] = first + i1 - v1;
        if (lane == 31) s_start[64] = first + i1;
        int total = t0 + t1;
        long long nvt = lane < n_warps ? s_nv[lane] : 0;
        double swt = 0.0, amt = lane < n_warps ? s_am[lane] : 0.0;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            total += __shfl_xor_sync(0xffffffffu, total, d);
            nvt += __shfl_xor_sync(0xffffffffu, nvt, d);
            amt = fmax(amt, __shfl_xor_sync(0xffffffffu, amt, d));
        }
        if (lane == 0) {
            for (int w = 0; w < n_warps; ++w) swt += s_sw[w];  // warp order
            info->n_visible = nvt;
            info->n_entries = total;
            info->sum_weights = swt;
            info->max_abs_dshift = amt;
        }
    }
    __syncthreads();
    for (int b = tid; b <= n_mu; b += nt) row_start[b] = s_start[b];  // s_start[n_mu] = the padded total
    for (int b = warp; b < n_mu; b += n_warps) {
        const double *row = sW + (size_t)b * Np;
        int pos = s_start[b];
        for (int j0 = 0; j0 < N; j0 += 32) {
            const int j = j0 + lane;
            const double W = j < N ? row[j] : 0.0;
            const unsigned m = __ballot_sync(0xffffffffu, W != 0.0);
            if (W != 0.0) {
                const int e = pos + __popc(m & ((1u << lane) - 1u));
                const double A = sA[j];
                ent32[e] = make_float2((float)A, (float)W);
                ent64[e] = make_double2(A, W);
            }
            pos += __popc(m);
        }
        if (lane == 0 && (s_cnt[b] & 1)) {
            ent32[pos] = make_float2(0.f, 0.f);
            ent64[pos] = make_double2(0.0, 0.0);
        }
    }
    if (!comp_Wp) return;
    // ---- pair tables of the composite-column form: (W[2p][b], W[2p+1][b]) as float2, the pair's shift factors, the
    // number of weight loads that cover its non-zero bins, and the exclusive prefix of the pairs' costs ---------------
    const int n_pairs = (N + 1) / 2;
    for (int k = tid; k < n_pairs * comp_stride; k += nt) {
        const int p = k / comp_stride, b = k - p * comp_stride;
        float2 w = make_float2(0.f, 0.f);
        if (b < n_mu) {
            w.x = (float)sW[(size_t)b * Np + 2 * p];
            if (2 * p + 1 < N) w.y = (float)sW[(size_t)b * Np + 2 * p + 1];
        }
        comp_Wp[k] = w;
    }
    for (int p = warp; p < n_pairs; p += n_warps) {
        const int j0 = 2 * p, j1 = 2 * p + 1;
        int hi = -1;
        for (int b0 = 0; b0 < n_mu; b0 += 32) {
            const int b = b0 + lane;
            const bool nz = b < n_mu && (sW[(size_t)b * Np + j0] != 0.0 || (j1 < N && sW[(size_t)b * Np + j1] != 0.0));
            const unsigned m = __ballot_sync(0xffffffffu, nz);
            if (m) hi = b0 + 31 - __clz(m);
        }
        if (lane == 0) s_cost[p] = (hi + 2) / 2;  // nl for now
    }
    __syncthreads();
    // exclusive scan of the costs, 32 * n_warps pairs per round (one round up to N = 2048)
    int carry = 0;
    for (int p0 = 0; p0 < n_pairs; p0 += nt) {
        const int p = p0 + tid;
        const int nl = p < n_pairs ? s_cost[p] : 0;
        const int c = p < n_pairs ? 8 * nl + comp::kPairCostBase : 0;
        int incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += u;
        }
        if (lane == 31) s_carry[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const int v = lane < n_warps ? s_carry[lane] : 0;
            int iw = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, iw, d);
                if (lane >= d) iw += u;
            }
            s_carry[lane] = iw - v;
            if (lane == 31) s_carry[32] = iw;
        }
        __syncthreads();
        if (p < n_pairs) {
            comp::PairHdr h;
            h.a0 = (float)sA[2 * p];
            h.a1 = 2 * p + 1 < N ? (float)sA[2 * p + 1] : 0.f;
            h.nl = nl;
            h.cost0 = carry + s_carry[warp] + incl - c;
            comp_hdr[p] = h;
        }
        carry += s_carry[32];
        __syncthreads();
    }
    if (tid == 0) {
        comp::PairHdr t;
        t.a0 = t.a1 = 0.f;
        t.nl = 0;
        t.cost0 = carry;
        comp_hdr[n_pairs] = t;
    }
}

// Per-cell form (SOAP_FORM_CELLS, and always under differential rotation, where the cells of a column no longer
// share a velocity): one entry per visible cell - the literal double loop of Alg. 1 - in the same layout, rows
// sorted by (column, row) so that neighbouring entries have nearly equal shifts.  The last CTA of geometry_kernel
// turns the per-(column, mu-bin) cell counts into row starts and per-column positions (one warp per mu-bin);
// write_cell_entries_kernel then writes the entries, one warp per column.
__device__ void build_cell_positions(int N, int n_mu, const int *colcnt, int *cellpos, int *row_start, float2 *ent32,
                                     double2 *ent64) {
    __shared__ int s_cnt[64];
    __shared__ int s_start[65];
    constexpr int kBatch = 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
    for (int b = warp; b < n_mu; b += n_warps) {
        int cnt = 0;
        for (int j0 = 0; j0 < N; j0 += 32 * kBatch) {
            int v[kBatch];
#pragma unroll
            for (int k = 0; k < kBatch; ++k) {
                const int j = j0 + 32 * k + lane;
                v[k] = j < N ? colcnt[(size_t)j * n_mu + b] : 0;
            }
#pragma unroll
            for (int k = 0; k < kBatch; ++k) cnt += v[k];
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, d);
        if (lane == 0) s_cnt[b] = cnt;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int off = 0;
        for (int b = 0; b < n_mu; ++b) {
            s_start[b] = off;
            off += (s_cnt[b] + 1) & ~1;
        }
        s_start[n_mu] = off;
    }
    __syncthreads();
    for (int b = threadIdx.x; b <= n_mu; b += blockDim.x) row_start[b] = s_start[b];
    for (int b = warp; b < n_mu; b += n_warps) {
        int run = s_start[b];
        for (int j0 = 0; j0 < N; j0 += 32) {
            const int j = j0 + lane;
            const int v = j < N ? colcnt[(size_t)j * n_mu + b] : 0;
            int incl = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            if (j < N) cellpos[(size_t)b * N + j] = run + incl - v;
            run += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (lane == 0 && (s_cnt[b] & 1)) {  // zero-weight pad entry: rows stay 16-byte aligned
            ent32[run] = make_float2(0.f, 0.f);
            ent64[run] = make_double2(0.0, 0.0);
        }
    }
}

// a1 + a2.  The fp64 geometry of a cell costs a few hundred instructions, so the cells are spread over the
// whole GPU: a CTA of 32 warps takes `cols_per_cta` columns, a warp takes one 32-row chunk of one column
// (or several, strided, when a column has more chunks than the CTA has warps per column).  Per column:
// every cell's (mu, w, v, bin), the shift factor a_j = D_j - 1 (all cells of a column share one velocity
// under solid-body rotation), the binned weights W[j][b] (per-warp partial sums added in warp order:
// deterministic) and the visible-cell count / weight sum.  The last CTA to finish compacts the binned
// weights into the entry list (build_binned_entries), so a1 + a2 are one launch.  `done` is zero on entry
// and is left zero.
__host__ __device__ inline int geom_warps_per_col(int N) {
    const int nc = (N + 31) / 32;
    return nc < kGeomWarps ? nc : kGeomWarps;
}
__host__ __device__ inline int geom_cols_per_cta(int N) { return kGeomWarps / geom_warps_per_col(N); }

struct GeomArgs {  // one star's geometry launch
    int N, mode, n_mu, cells, comp_stride, fin_smem, n_ctas, pad;
    Rotation rot;
    double u1, u2;
    MuCentres mu_centres;
    double *mu_out, *w_out, *vel_out;
    int *bin_out;
    double *col_a, *Wbin /*[N][n_mu]*/, *col_sumw;
    int *col_nvis;
    float2 *ent32;
    double2 *ent64;
    int *row_start;
    DevInfo *info;
    unsigned int *done;
    int *colcnt /*[N][n_mu]*/, *cellpos /*[n_mu][N], per-cell form only*/;
    float2 *comp_Wp /*composite form: [ceil(N/2)][comp_stride], or nullptr*/;
    comp::PairHdr *comp_hdr;
};
static_assert(sizeof(GeomArgs) % 8 == 0, "copied to shared memory in 8-byte words");

// `one`: a single star (many == nullptr).  Batch (soap_batch_disk_geometry): `many` = DEVICE [n_stars] arguments, `cta0` =
// DEVICE [n_stars + 1] first CTA of every star; every star keeps its own last-CTA ticket.
// dynamic shared memory = the largest fin_smem_bytes(N, n_mu) of the stars with fin_smem set.
__global__ void __launch_bounds__(32 * kGeomWarps)
geometry_kernel(const GeomArgs one, const GeomArgs *__restrict__ many, const int *__restrict__ cta0, int n_stars) {
    extern __shared__ __align__(16) unsigned char geom_dyn[];
    __shared__ double s_W[kGeomWarps][64];
    __shared__ int s_Cn[kGeomWarps][64];
    __shared__ double s_mu[64];
    __shared__ double s_sum[kGeomWarps];
    __shared__ int s_nvis[kGeomWarps];
    __shared__ int s_last, s_first;
    __shared__ GeomArgs s_a;
    {
        int star = 0, first = 0;
        if (many) {
            int lo = 0, hi = n_stars - 1;  // last star with cta0[s] <= blockIdx.x
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (__ldcg(&cta0[mid]) <= (int)blockIdx.x) lo = mid;
                else hi = mid - 1;
            }
            star = lo;
            first = __ldcg(&cta0[lo]);
        }
        const unsigned long long *src = reinterpret_cast<const unsigned long long *>(many ? many + star : &one);
        unsigned long long *dst = reinterpret_cast<unsigned long long *>(&s_a);
        for (int k = threadIdx.x; k < (int)(sizeof(GeomArgs) / 8); k += blockDim.x) dst[k] = src[k];
        if (threadIdx.x == 0) s_first = first;
    }
    __syncthreads();
    const int N = s_a.N, mode = s_a.mode, n_mu = s_a.n_mu;
    const Rotation rot = s_a.rot;
    const double u1 = s_a.u1, u2 = s_a.u2;
    const MuCentres &mu_centres = s_a.mu_centres;
    double *__restrict__ mu_out = s_a.mu_out, *__restrict__ w_out = s_a.w_out, *__restrict__ vel_out = s_a.vel_out;
    int *__restrict__ bin_out = s_a.bin_out;
    double *__restrict__ col_a = s_a.col_a, *__restrict__ Wbin = s_a.Wbin, *__restrict__ col_sumw = s_a.col_sumw;
    int *__restrict__ col_nvis = s_a.col_nvis, *__restrict__ colcnt = s_a.colcnt;
    unsigned int *__restrict__ done = s_a.done;
    const int bid = (int)blockIdx.x - s_first;  // this star's CTA number
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    trigger_dependents();  // the quiet launch that follows may stage its spectra while this kernel runs (ptx_helpers.cuh)
    for (int b = threadIdx.x; b < n_mu; b += blockDim.x) s_mu[b] = mu_centres.v[b];
    for (int b = lane; b < 64; b += 32) {
        s_W[warp][b] = 0.0;
        s_Cn[warp][b] = 0;
    }
    __syncthreads();
    const int wpc = geom_warps_per_col(N), cpc = kGeomWarps / wpc;
    const int cl = warp / wpc, chunk = warp - cl * wpc;  // local column, first chunk
    const int j = bid * cpc + cl;
    double sum = 0.0;
    int nvis = 0;
    if (cl < cpc && j < N) {
        geometry_chunks(j, chunk, wpc, N, rot, u1, u2, n_mu, s_mu, s_W[warp], s_Cn[warp], mu_out, w_out, vel_out, bin_out, sum, nvis);
        // the column's shift factor (solid body; with differential rotation the per-cell form is used instead): by the
        // warp of the column's first chunk, whose cells are mostly off the disk - it has time to spare
        if (chunk == 0 && lane == 0)
            col_a[j] = doppler_minus_one(__dmul_rn(__dmul_rn(cell_coord(j, N), rot.vsini), rot.sini), mode);
    }
    if (lane == 0) {
        s_sum[warp] = sum;
        s_nvis[warp] = nvis;
    }
    __syncthreads();
    if (warp < cpc) {  // warp `warp` finishes local column `warp`
        const int jj = bid * cpc + warp;
        if (jj < N) {
            for (int b = lane; b < n_mu; b += 32) {
                double W = 0.0;
                int C = 0;
                for (int k = 0; k < wpc; ++k) {
                    W += s_W[warp * wpc + k][b];
                    C += s_Cn[warp * wpc + k][b];
                }
                Wbin[(size_t)jj * n_mu + b] = W;
                colcnt[(size_t)jj * n_mu + b] = C;
            }
            if (lane == 0) {
                double sw = 0.0;
                int nv = 0;
                for (int k = 0; k < wpc; ++k) {
                    sw += s_sum[warp * wpc + k];
                    nv += s_nvis[warp * wpc + k];
                }
                col_sumw[jj] = sw;
                col_nvis[jj] = nv;
            }
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(done, 1u) == (unsigned)s_a.n_ctas - 1u) ? 1 : 0;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x == 0) *done = 0;
    if (s_a.fin_smem) {
        finalize_columns_smem(N, n_mu, col_a, Wbin, col_sumw, col_nvis, s_a.ent32, s_a.ent64, s_a.row_start, s_a.info, s_a.comp_Wp,
                              s_a.comp_stride, s_a.comp_hdr, geom_dyn);
    } else {
        build_binned_entries(N, n_mu, col_a, Wbin, col_sumw, col_nvis, s_a.ent32, s_a.ent64, s_a.row_start, s_a.info);
        if (s_a.comp_Wp) {  // pair tables of the composite-column form (composite.cuh)
            __syncthreads();
            comp::build_composite_tables(N, n_mu, col_a, Wbin, s_a.comp_Wp, s_a.comp_stride, s_a.comp_hdr);
        }
    }
    if (s_a.cells) {  // per-cell form: the entry list is rebuilt by write_cell_entries_kernel at these positions
        __syncthreads();
        build_cell_positions(N, n_mu, colcnt, s_a.cellpos, s_a.row_start, s_a.ent32, s_a.ent64);
    }
}

// One warp per column: writes the column's cells as entries (a_c, w_c), a_c = D_c - 1 from the cell's own velocity,
// at cellpos[bin][column] + rank among the column's earlier cells of that bin (row order).
constexpr int kCellWarps = 8;
__global__ void __launch_bounds__(32 * kCellWarps)
write_cell_entries_kernel(int N, int n_mu, int mode, const double *__restrict__ vel, const double *__restrict__ w,
                          const int *__restrict__ bin, const int *__restrict__ cellpos, float2 *__restrict__ ent32,
                          double2 *__restrict__ ent64) {
    __shared__ int s_pos[kCellWarps][64];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int j = blockIdx.x * kCellWarps + warp;
    if (j >= N) return;
    for (int b = lane; b < n_mu; b += 32) s_pos[warp][b] = cellpos[(size_t)b * N + j];
    __syncwarp();
    for (int i0 = 0; i0 < N; i0 += 32) {
        const int i = i0 + lane;
        const size_t c = (size_t)j * N + (i < N ? i : N - 1);
        const int b = i < N ? bin[c] : -1;
        const double v = vel[c], wc = w[c];
        const unsigned same = __match_any_sync(0xffffffffu, b);
        int e = 0;
        if (b >= 0) e = s_pos[warp][b] + __popc(same & ((1u << lane) - 1u));
        __syncwarp();
        if (b >= 0 && lane == __ffs(same) - 1) s_pos[warp][b] += __popc(same);
        __syncwarp();
        if (b >= 0) {
            const double a = doppler_minus_one(v, mode);
            ent32[e] = make_float2((float)a, (float)wc);
            ent64[e] = make_double2(a, wc);
        }
    }
}

}  // namespace soap
