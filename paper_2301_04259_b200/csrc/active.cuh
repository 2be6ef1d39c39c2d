// a4 of SURVEY section 8: per-phase active map and compaction (InfoMap of Alg. 5).
//
// The paper rewrites an N x N type map on the device at every timestamp.  Here the map is never
// materialised.  One thread-block cluster of 8 CTAs per (star, phase); CTA `rank` owns an eighth of the list of
// columns the phase's regions can reach.  A warp walks a column, decides each cell's type by spherical
// angular distance with list-order override, and bins the covered cells by (kind, mu-bin) - all cells of a
// column share one velocity - into shared memory.  The CTAs push their per-segment entry counts into each
// other's shared memory (distributed shared memory), so that each can compact its non-zero bins of every
// (kind, mu-bin) segment behind those of the lower ranks: the entry list the shift-interpolate-accumulate
// kernel consumes is in column order.  Rank 0 writes the phase's job list and its job / entry counts; the
// active launch takes the phases heaviest first by the latter (sia_f32.cuh).
// One launch, no scratch to zero, no floating-point atomics (every sum has a fixed order).
// Kinds: 0 = quiet row of a covered cell (weight -w), 1 = spot row, 2 = facula row (weight +w LB_t(mu)).
// Effects form (the three outputs of Eq. 1-3 from one pass, sia_f32.cuh): the quiet rows are kept per region type -
// kind 0 = quiet row under a spot, 3 = under a facula - and, for a region type whose limb-brightening law differs from 1
// (PrepArgs::lb_types), kinds 4, 5 = quiet row with weight +w LB_t(mu) and 6, 7 = spot / facula row with weight +w
// (flux-only and CB-only use them).
#pragma once
#include <cstdint>
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include "geometry.cuh"
#include "ptx_helpers.cuh"

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

struct ActiveJob {  // one job of a phase's list: <= kActiveJobCap consecutive entries of one segment
    int begin;      // first entry (global index, even)
    int count;      // entries, 1..kActiveJobCap
    int kind, row;
};
constexpr int kActiveJobCap = 128;      // == f32::kJobCap
constexpr int kPrepCluster = 8;         // CTAs per phase (portable cluster size)
constexpr int kPrepThreads = 512;       // 16 warps per CTA (active_prepare_kernel: THREADS, see below)
constexpr int kPrepChunks = 4;          // 32-row chunks of a column whose cell data is loaded together

struct ActiveCounters {  // device-resident
    int item_next, item_ctas_done;      // hand-out of (phase, tile) items in the active launch (self-resetting)
    int overflow;                       // per-cell form: a phase's entry pool was too small (cannot happen with the host's bound)
    int pad;
};

struct PrepArgs {
    int N, n_regions, n_mu, seg_cap, chunk_cols, job_cap, n_phases;
    int n_kinds;              // 3; effects form: 4 (both limb-brightening laws are 1) or 8
    int lb_types;             // effects form with 8 kinds: bit t = region type t has a limb-brightening law other than 1
    const RegionAtPhase *rp;  // [n_phases][n_regions]
    const double *mu, *w, *col_a;
    const int *bin;
    LbCoef lb;
    void *ent;                // [n_phases * n_kinds n_mu][seg_cap] of EntT
    int *seg_count;           // [n_phases * n_kinds n_mu]
    int *n_active;            // [n_phases] covered cells
    ActiveJob *jobs;          // [n_phases][job_cap]
    int *n_jobs, *work;       // [n_phases] each: jobs and entries of the phase (the active launch takes the heaviest first)
    ActiveCounters *counters;
    // per-cell form (differential rotation / SOAP_FORM_CELLS): every covered cell is an entry with its own shift
    const double *vel;        // [N*N] cell velocities
    int mode;                 // doppler_mode
    int pool_cap;             // entries a phase's pool can hold (even); ent = [n_phases][pool_cap]
};

constexpr int kPrepRegSmem = 256;       // regions of a phase held in shared memory (more: read from global memory)
struct PrepLayout {  // dynamic shared memory of active_prepare_kernel (byte offsets, each a multiple of 16)
    size_t cnt_off, cols_off, reg_off, bytes;
};
__host__ __device__ inline PrepLayout prep_layout(int n_mu, int chunk_cols, int N, int n_regions, int n_kinds = 3) {
    PrepLayout l;
    l.cnt_off = ((size_t)n_kinds * n_mu * chunk_cols * sizeof(double) + 15) & ~(size_t)15;
    l.cols_off = l.cnt_off + (((size_t)kPrepCluster * n_kinds * n_mu * sizeof(int) + 15) & ~(size_t)15);
    l.reg_off = l.cols_off + (((size_t)N * sizeof(int) + 15) & ~(size_t)15);
    l.bytes = l.reg_off + (size_t)(n_regions <= kPrepRegSmem ? n_regions : 0) * sizeof(RegionAtPhase) + 16;
    return l;
}
__host__ __device__ inline size_t prep_smem_bytes(int n_mu, int chunk_cols, int N, int n_regions, int n_kinds = 3) {
    return prep_layout(n_mu, chunk_cols, N, n_regions, n_kinds).bytes;
}


// The regions that can reach column x (|x - x_r| <= chord), in list order, gathered by one warp into cand[] so that
// the per-cell membership loop visits only them (hundreds of regions: a column meets a few tens).  Returns their
// number, or -1 when they do not fit (the caller then walks the whole list); [ylo, yhi] bounds the rows they reach.
constexpr int kCandCap = 128;
__device__ __forceinline__ int column_candidates(const RegionAtPhase *reg, int n_regions, double x, int lane, int *cand,
                                                 double &ylo, double &yhi) {
    int n = 0;
    bool fits = true;
    ylo = 2.0;
    yhi = -2.0;
    __syncwarp();
    for (int r0 = 0; r0 < n_regions; r0 += 32) {
        const int r = r0 + lane;
        bool hit = false;
        if (r < n_regions && reg[r].type != 0) {
            const double ch = reg[r].chord * (1.0 + 1e-9) + 1e-12;
            if (fabs(x - reg[r].xr) <= ch) {
                hit = true;
                ylo = fmin(ylo, reg[r].yr - ch);
                yhi = fmax(yhi, reg[r].yr + ch);
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        const int k = n + __popc(m & ((1u << lane) - 1u));
        if (hit && k < kCandCap) cand[k] = r;
        n += __popc(m);
        fits = fits && n <= kCandCap;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        ylo = fmin(ylo, __shfl_xor_sync(0xffffffffu, ylo, d));
        yhi = fmax(yhi, __shfl_xor_sync(0xffffffffu, yhi, d));
    }
    __syncwarp();
    return fits ? n : -1;
}

// grid = n_phases * kPrepCluster, block = THREADS, cluster = kPrepCluster CTAs;
// dynamic shared memory = prep_smem_bytes(n_mu, chunk_cols, n_regions) with chunk_cols >= ceil(N / kPrepCluster).
// Batch form (soap_batch_active_timeseries): `many` = DEVICE [n_stars] arguments, `phase0` = DEVICE [n_stars + 1] first
// cluster (phase) of every star; cluster c serves phase c - phase0[s] of the star s that holds it.  many == nullptr: `one`.
//
// The kernel is latency-sized (a few thousand cells per phase), so its structure follows its dependent steps, not its
// arithmetic: (1) arguments, the phase's regions -> shared memory, accumulators zeroed; (2) the columns any region can
// reach, compacted into a list that the CTAs of the cluster share out evenly (two far-apart regions do not leave half
// of the CTAs idle); (3) bin; (4) per-segment counts PUSHED into every CTA of the cluster through distributed shared
// memory, one cluster barrier; (5) compaction behind the lower ranks' entries; rank 0 writes the job list (parallel
// scan over the segments).  No CTA waits for another phase: the order in which the shift-interpolate-accumulate launch
// takes the phases (heaviest first) is derived there from work[] (sia_f32.cuh).
// THREADS: 512 when all the clusters of the launch are resident at once (the launch is then as long as its slowest cluster:
// the more warps share a phase's columns the better); 256 beyond that - half of the warps of a cluster wait at its barriers
// at any time (load imbalance between columns), and twice the clusters per SM fill the idle issue slots (C4: 99 -> 67 us).
// `inl` (K > 0): the region centres of a single star's call travel as a kernel argument - [n_phases][n_regions], at most K -
// so that the call needs no host -> device copy at all; K == 0: they are read from a.rp.
template <int K>
struct InlineRegions {
    RegionAtPhase r[K > 0 ? K : 1];
};
constexpr int kInlineRegions = 192;  // 9 KB of kernel arguments

template <typename EntT, int K, int THREADS>
__global__ void __cluster_dims__(kPrepCluster, 1, 1) __launch_bounds__(THREADS)
active_prepare_kernel(const PrepArgs one, const PrepArgs *__restrict__ many, const int *__restrict__ phase0, int n_stars,
                      const __grid_constant__ InlineRegions<K> inl) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char prep_smem[];
    __shared__ PrepArgs s_args;
    __shared__ int s_phase;
    __shared__ int s_cand[THREADS / 32][kCandCap];  // per warp: regions that can reach its column
    __shared__ int s_misc[4];                            // reachable columns, covered cells of this CTA
    __shared__ int s_cov[kPrepCluster];                  // rank 0: covered cells of every CTA (pushed)
    __shared__ int s_wsum[THREADS / 32 + 1], s_wjobs[THREADS / 32 + 1];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, n_warps = THREADS / 32;
    // every CTA of the cluster must be running before its shared memory is written remotely: arrive now, wait in (4)
    asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
    // (launched with programmatic stream serialization: the geometry this kernel reads is complete after the wait)
    trigger_dependents();
    grid_dependency_wait();
    if (tid == 0) {
        const int c = blockIdx.x / kPrepCluster;
        if (many) {
            int lo = 0, hi = n_stars - 1;  // last star with phase0[s] <= c
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (__ldcg(&phase0[mid]) <= c) lo = mid;
                else hi = mid - 1;
            }
            s_args = many[lo];
            s_phase = c - __ldcg(&phase0[lo]);
        } else {
            s_args = one;
            s_phase = c;
        }
        s_misc[0] = 0;
        s_misc[2] = 0;
    }
    __syncthreads();
    const PrepArgs &a = s_args;
    const int n_seg = a.n_kinds * a.n_mu, N = a.N, cc = a.chunk_cols;
    const PrepLayout lay = prep_layout(a.n_mu, cc, N, a.n_regions, a.n_kinds);
    double *WDs = reinterpret_cast<double *>(prep_smem);                  // [n_seg][cc]: this CTA's columns
    int *cnt_all = reinterpret_cast<int *>(prep_smem + lay.cnt_off);      // [kPrepCluster][n_seg] entries of every CTA (pushed)
    int *s_cols = reinterpret_cast<int *>(prep_smem + lay.cols_off);      // [N] reachable columns, ascending
    const int n_reg_sm = a.n_regions <= kPrepRegSmem ? a.n_regions : 0;
    RegionAtPhase *s_reg = reinterpret_cast<RegionAtPhase *>(prep_smem + lay.reg_off);  // [n_reg_sm]
    const int p = s_phase;
    const int rank = (int)cluster.block_rank();
    const RegionAtPhase *greg = (K > 0 ? inl.r : a.rp) + (size_t)p * a.n_regions;
    EntT *ent = static_cast<EntT *>(a.ent) + (size_t)p * n_seg * a.seg_cap;

    // ---- (1) regions -> shared memory (16-byte copies), accumulators zeroed ----------------------------------------------
    {
        const uint4 *src = reinterpret_cast<const uint4 *>(greg);
        uint4 *dst = reinterpret_cast<uint4 *>(s_reg);
        for (int k = tid; k < n_reg_sm * (int)(sizeof(RegionAtPhase) / 16); k += THREADS) dst[k] = K > 0 ? src[k] : __ldcg(&src[k]);
        for (int k = tid; k < n_seg * cc; k += THREADS) WDs[k] = 0.0;
    }
    __syncthreads();
    const RegionAtPhase *reg = n_reg_sm ? s_reg : greg;
    // ---- (2) the columns some region of this phase can reach (conservative: chord bound, slightly inflated) -------------
    for (int j0 = 0; j0 < N; j0 += THREADS) {
        const int j = j0 + tid;
        bool hit = false;
        if (j < N) {
            const double x = cell_coord(j, N);
            for (int r = 0; r < a.n_regions && !hit; ++r)
                hit = reg[r].type != 0 && fabs(x - reg[r].xr) <= reg[r].chord * (1.0 + 1e-9) + 1e-12;
        }
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (lane == 0) s_wsum[warp] = __popc(m);
        __syncthreads();
        int before = s_misc[0];
        for (int w = 0; w < warp; ++w) before += s_wsum[w];
        if (hit) s_cols[before + __popc(m & ((1u << lane) - 1u))] = j;
        __syncthreads();
        if (tid == 0) {
            int t = 0;
            for (int w = 0; w < n_warps; ++w) t += s_wsum[w];
            s_misc[0] += t;
        }
        __syncthreads();
    }
    const int n_reach = s_misc[0];
    const int per = (n_reach + kPrepCluster - 1) / kPrepCluster;  // columns per CTA, <= cc
    const int k0c = rank * per;
    const int cols = max(0, min(per, n_reach - k0c));
    if (n_reach == 0 && a.n_phases > 1) {
        // No region of this phase faces the observer (every CTA of the cluster sees the same list): an empty phase.
        // Rank 0 records it; nothing is binned, exchanged or compacted.
        if (rank != 0) return;
        for (int s = tid; s < n_seg; s += THREADS) a.seg_count[p * n_seg + s] = 0;
        if (tid == 0) {
            a.n_jobs[p] = 0;
            a.work[p] = 0;
            a.n_active[p] = 0;
        }
        return;
    }
    // ---- (3) bin: one warp per column, lanes over the rows (coalesced) -------------------------------------------------
    for (int kc = warp; kc < cols; kc += n_warps) {
        const int j = s_cols[k0c + kc];
        const double x = cell_coord(j, N);
        double ylo, yhi;
        const int n_cand = column_candidates(reg, a.n_regions, x, lane, s_cand[warp], ylo, yhi);
        const int n_loop = n_cand < 0 ? a.n_regions : n_cand;
        if (ylo > yhi) continue;
        int i_lo = (int)floor((ylo + 1.0) * 0.5 * N - 0.5) - 1;
        int i_hi = (int)ceil((yhi + 1.0) * 0.5 * N - 0.5) + 1;
        i_lo = max(i_lo, 0);
        i_hi = min(i_hi, N - 1);
        double *col = WDs + kc;
        int count = 0;
        for (int i00 = i_lo; i00 <= i_hi; i00 += 32 * kPrepChunks) {
            // all loads of up to kPrepChunks chunks are issued before any is used: one memory round trip
            int bb[kPrepChunks];
            double mm[kPrepChunks], ww[kPrepChunks];
#pragma unroll
            for (int k = 0; k < kPrepChunks; ++k) {
                const int i = i00 + 32 * k + lane;
                const bool in = i <= i_hi;
                const size_t c = (size_t)j * N + (in ? i : i_hi);
                bb[k] = in ? a.bin[c] : -1;  // hidden cells: bin -1, mu 0, w 0
                mm[k] = a.mu[c];
                ww[k] = a.w[c];
            }
#pragma unroll
            for (int k = 0; k < kPrepChunks; ++k) {
                if (i00 + 32 * k > i_hi) break;
                const int i = i00 + 32 * k + lane;
                const int b = bb[k];
                const double m = mm[k];
                int t = 0;
                double wc = 0.0, wl = 0.0;
                if (b >= 0) {
                    const double y = cell_coord(i, N);
                    for (int q = 0; q < n_loop; ++q) {  // list order: the last covering region wins
                        const int r = n_cand < 0 ? q : s_cand[warp][q];
                        if (reg[r].type == 0) continue;
                        const double dot = __dadd_rn(__dadd_rn(__dmul_rn(x, reg[r].xr), __dmul_rn(y, reg[r].yr)),
                                                     __dmul_rn(m, reg[r].zr));
                        if (dot >= reg[r].cos_alpha) t = reg[r].type;
                    }
                    if (t != 0) {
                        wc = ww[k];
                        wl = wc * (a.lb.c[t][0] + a.lb.c[t][1] * m + a.lb.c[t][2] * m * m);
                    }
                }
                // cells of equal (mu-bin, type) are contiguous in a column: segmented scans, added in row order
                const int key = (t != 0) ? (b * 4 + t) : -1;
                int start;
                bool tail;
                const double seg_w = warp_segmented_scan(wc, key, lane, start, tail);
                const double seg_wl = warp_segmented_scan(wl, key, lane, start, tail);
                unsigned tails = __ballot_sync(0xffffffffu, tail && t != 0);
                while (tails) {
                    const int l = __ffs(tails) - 1;
                    if (lane == l) {
                        const int kq = (a.n_kinds > 3 && t == 2) ? 3 : 0;  // effects form: quiet rows per region type
                        col[(size_t)(kq * a.n_mu + b) * cc] += seg_w;
                        col[(size_t)(t * a.n_mu + b) * cc] += seg_wl;
                        if (a.n_kinds == 8 && ((a.lb_types >> t) & 1)) {
                            col[(size_t)((3 + t) * a.n_mu + b) * cc] += seg_wl;
                            col[(size_t)((5 + t) * a.n_mu + b) * cc] += seg_w;
                        }
                    }
                    __syncwarp();
                    tails &= tails - 1;
                }
                count += __popc(__ballot_sync(0xffffffffu, t != 0));
            }
        }
        if (lane == 0 && count) atomicAdd(&s_misc[2], count);  // integer: order-independent
    }
    __syncthreads();
    // ---- (4) this CTA's entries per segment, pushed to every CTA of the cluster -------------------------------------------
    asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
    for (int s = warp; s < n_seg; s += n_warps) {
        const double *src = WDs + (size_t)s * cc;
        int c = 0;
        for (int k0 = 0; k0 < cols; k0 += 32) {
            const int k = k0 + lane;
            c += __popc(__ballot_sync(0xffffffffu, k < cols && src[k] != 0.0));
        }
        if (lane < kPrepCluster) cluster.map_shared_rank(cnt_all, lane)[rank * n_seg + s] = c;
    }
    if (tid == 0) cluster.map_shared_rank(s_cov, 0)[rank] = s_misc[2];
    cluster.sync();  // every count has arrived; nobody touches another CTA's shared memory after this
    // ---- (5) compact: one warp per segment, this CTA's columns in order, behind the lower ranks' entries -------------
    for (int s = warp; s < n_seg; s += n_warps) {
        const int sk = s / a.n_mu;
        const double sign = (sk == 0 || (sk == 3 && a.n_kinds > 3)) ? -1.0 : 1.0;
        const double *src = WDs + (size_t)s * cc;
        int ps = 0;
        for (int r = 0; r < rank; ++r) ps += cnt_all[r * n_seg + s];
        EntT *dst = ent + (size_t)s * a.seg_cap;
        for (int k0 = 0; k0 < cols; k0 += 32) {
            const int k = k0 + lane;
            const double W = (k < cols) ? src[k] : 0.0;
            const unsigned m = __ballot_sync(0xffffffffu, W != 0.0);
            if (W != 0.0) {
                EntT e;
                e.x = (decltype(e.x))a.col_a[s_cols[k0c + k]];
                e.y = (decltype(e.y))(sign * W);
                dst[ps + __popc(m & ((1u << lane) - 1u))] = e;
            }
            ps += __popc(m);
        }
    }
    if (rank != 0) return;
    // ---- rank 0 finalises the phase: pad odd segments, counts, job list (kinds 1, 2, then 0).  Thread t takes the t-th
    // segment of the job order; jobs are numbered by a block-wide exclusive scan of the segments' job counts.
    for (int t0 = 0, jobs_before = 0, work_sum = 0; t0 < n_seg || t0 == 0; t0 += THREADS) {
        const int t = t0 + tid;
        int s = 0, c = 0;
        if (t < n_seg) {
            s = t + a.n_mu;
            if (s >= n_seg) s -= n_seg;
            for (int r = 0; r < kPrepCluster; ++r) c += cnt_all[r * n_seg + s];
            if (c & 1) {  // zero-weight pad entry: every job's entry block stays a multiple of 16 bytes
                EntT z;
                z.x = 0;
                z.y = 0;
                ent[(size_t)s * a.seg_cap + c] = z;
            }
            a.seg_count[p * n_seg + s] = c;
        }
        const int nj = (c + kActiveJobCap - 1) / kActiveJobCap;
        int incl = nj, wsum = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += u;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) wsum += __shfl_xor_sync(0xffffffffu, wsum, d);
        if (lane == 31) s_wjobs[warp] = incl;
        if (lane == 0) s_wsum[warp] = wsum;
        __syncthreads();
        int k = jobs_before + incl - nj;
        for (int w = 0; w < warp; ++w) k += s_wjobs[w];
        for (int o = 0; o < c; o += kActiveJobCap) {
            ActiveJob jb;
            jb.begin = (p * n_seg + s) * a.seg_cap + o;  // fits: host checks n_phases * n_kinds n_mu * seg_cap < 2^31
            jb.count = min(kActiveJobCap, c - o);
            jb.kind = s / a.n_mu;
            jb.row = s - jb.kind * a.n_mu;
            a.jobs[(size_t)p * a.job_cap + k++] = jb;
        }
        for (int w = 0; w < n_warps; ++w) {
            jobs_before += s_wjobs[w];
            work_sum += s_wsum[w];
        }
        __syncthreads();
        if (t0 + THREADS >= n_seg && tid == 0) {
            int covered = 0;
            for (int r = 0; r < kPrepCluster; ++r) covered += s_cov[r];
            a.n_jobs[p] = jobs_before;
            a.work[p] = work_sum;
            a.n_active[p] = covered;
        }
    }
}

// Walks column j of one phase: calls f(c, b, t, mu, w) for every lane of every 32-row chunk the regions can reach
// (warp-uniform number of calls; t = 0 for cells no region covers, b = -1 for hidden cells).
template <typename F>
__device__ __forceinline__ void walk_column(const PrepArgs &a, const RegionAtPhase *reg, int j, int lane, int *cand, F &&f) {
    const int N = a.N;
    const double x = cell_coord(j, N);
    double ylo, yhi;
    const int n_cand = column_candidates(reg, a.n_regions, x, lane, cand, ylo, yhi);
    const int n_loop = n_cand < 0 ? a.n_regions : n_cand;
    if (ylo > yhi) return;
    int i_lo = (int)floor((ylo + 1.0) * 0.5 * N - 0.5) - 1;
    int i_hi = (int)ceil((yhi + 1.0) * 0.5 * N - 0.5) + 1;
    i_lo = max(i_lo, 0);
    i_hi = min(i_hi, N - 1);
    for (int i0 = i_lo; i0 <= i_hi; i0 += 32) {
        const int i = i0 + lane;
        const bool in = i <= i_hi;
        const size_t c = (size_t)j * N + (in ? i : i_hi);
        const int b = in ? a.bin[c] : -1;
        const double m = a.mu[c], wc = a.w[c];
        int t = 0;
        if (b >= 0) {
            const double y = cell_coord(i, N);
            for (int q = 0; q < n_loop; ++q) {  // list order: the last covering region wins
                const int r = n_cand < 0 ? q : cand[q];
                if (reg[r].type == 0) continue;
                const double dot =
                    __dadd_rn(__dadd_rn(__dmul_rn(x, reg[r].xr), __dmul_rn(y, reg[r].yr)), __dmul_rn(m, reg[r].zr));
                if (dot >= reg[r].cos_alpha) t = reg[r].type;
            }
        }
        f(c, b, t, m, wc);
    }
}

// a4, per-cell form: the same cluster-per-phase structure as active_prepare_kernel, but every covered cell
// becomes its own pair of entries (a_c, -w) in the quiet segment of its mu-bin and (a_c, +w LB_t(mu)) in its
// kind's segment, because under differential rotation the cells of a column no longer share a
// velocity.  Two passes over the columns (count, then write) with the per-(segment, column) counts in shared
// memory; a phase's segments are packed back to back, in job order, in the phase's pool ent[p][pool_cap].
// Within a segment the entries are in (column, row) order: neighbouring entries have nearly equal shifts.
// dynamic shared memory = prep_cells_smem_bytes(n_mu, chunk_cols).
__host__ __device__ inline size_t prep_cells_smem_bytes(int n_mu, int chunk_cols) {
    return (size_t)3 * n_mu * chunk_cols * sizeof(int) + (size_t)4 * 3 * n_mu * sizeof(int) + 64;
}

template <typename EntT>
__global__ void __cluster_dims__(kPrepCluster, 1, 1) __launch_bounds__(kPrepThreads)
active_prepare_cells_kernel(const PrepArgs a) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char prep_smem[];
    const int n_seg = 3 * a.n_mu, N = a.N, cc = a.chunk_cols;
    __shared__ int s_cand[kPrepThreads / 32][kCandCap];  // per warp: regions that can reach its column
    int *cntc = reinterpret_cast<int *>(prep_smem);  // [n_seg][cc]: entries per (segment, column); then running offsets
    int *cnt = cntc + (size_t)n_seg * cc;            // [n_seg] entries of this CTA (read by the others)
    int *off = cnt + n_seg;                          // [n_seg] pool position of this CTA's block of the segment
    int *tot = off + n_seg;                          // [n_seg] entries of the whole phase
    int *base = tot + n_seg;                         // [n_seg] pool position of the segment
    int *s_misc = base + n_seg;                      // j_lo, j_hi, covered cells of this CTA
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, n_warps = kPrepThreads / 32;
    const int p = blockIdx.x / kPrepCluster;
    const int rank = (int)cluster.block_rank();
    const RegionAtPhase *reg = a.rp + (size_t)p * a.n_regions;
    EntT *pool = static_cast<EntT *>(a.ent) + (size_t)p * a.pool_cap;

    if (tid == 0) {
        s_misc[0] = N;
        s_misc[1] = -1;
        s_misc[2] = 0;
        s_misc[3] = 0;
    }
    __syncthreads();
    for (int r = tid; r < a.n_regions; r += kPrepThreads) {
        if (reg[r].type == 0) continue;
        const double ch = reg[r].chord * (1.0 + 1e-9) + 1e-12;
        int jl = (int)floor((reg[r].xr - ch + 1.0) * 0.5 * N - 0.5) - 1;
        int jh = (int)ceil((reg[r].xr + ch + 1.0) * 0.5 * N - 0.5) + 1;
        atomicMin(&s_misc[0], max(jl, 0));
        atomicMax(&s_misc[1], min(jh, N - 1));
    }
    __syncthreads();
    const int j_lo = s_misc[0], j_hi = s_misc[1];
    const int per = (j_hi >= j_lo) ? (j_hi - j_lo + kPrepCluster) / kPrepCluster : 0;
    const int c0 = j_lo + rank * per;
    const int cols = max(0, min(per, j_hi + 1 - c0));
    for (int s = warp; s < n_seg; s += n_warps)
        for (int k = lane; k < cols; k += 32) cntc[(size_t)s * cc + k] = 0;
    __syncthreads();
    // ---- pass 1: count the covered cells per (segment, column) ------------------------------------------------
    for (int j = c0 + warp; j < c0 + cols; j += n_warps) {
        int *col = cntc + (j - c0);
        int count = 0;
        walk_column(a, reg, j, lane, s_cand[warp], [&](size_t, int b, int t, double, double) {
            // the quiet segment of a mu-bin collects the covered cells of every type, the kind segments one type each
            const unsigned same0 = __match_any_sync(0xffffffffu, t != 0 ? b : -1);
            const unsigned same = __match_any_sync(0xffffffffu, t != 0 ? b * 4 + t : -1);
            if (t != 0 && lane == __ffs(same0) - 1) col[(size_t)b * cc] += __popc(same0);  // one lane per distinct key
            if (t != 0 && lane == __ffs(same) - 1) col[(size_t)(t * a.n_mu + b) * cc] += __popc(same);
            __syncwarp();
            count += __popc(__ballot_sync(0xffffffffu, t != 0));
        });
        if (lane == 0 && count) atomicAdd(&s_misc[2], count);
    }
    __syncthreads();
    // ---- per segment: exclusive scan over this CTA's columns, CTA total ----------------------------------------
    for (int s = warp; s < n_seg; s += n_warps) {
        int *row = cntc + (size_t)s * cc;
        int run = 0;
        for (int k0 = 0; k0 < cols; k0 += 32) {
            const int k = k0 + lane;
            const int v = k < cols ? row[k] : 0;
            int incl = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            if (k < cols) row[k] = run + incl - v;
            run += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (lane == 0) cnt[s] = run;
    }
    cluster.sync();
    for (int s = tid; s < n_seg; s += kPrepThreads) {
        int before = 0, all = 0;
        for (int r = 0; r < kPrepCluster; ++r) {
            const int c = cluster.map_shared_rank(cnt, r)[s];
            before += r < rank ? c : 0;
            all += c;
        }
        off[s] = before;
        tot[s] = all;
    }
    int covered = 0;
    if (rank == 0 && tid == 0)
        for (int r = 0; r < kPrepCluster; ++r) covered += cluster.map_shared_rank(s_misc, r)[2];
    cluster.sync();  // no CTA goes on to change cnt / s_misc while they are being read
    // segment positions in the pool: job order (kinds 1, 2, then 0), each padded to an even length
    if (warp == 0) {
        const int per_lane = (n_seg + 31) / 32;
        const int ss0 = min(n_seg, lane * per_lane), ss1 = min(n_seg, ss0 + per_lane);
        int mine = 0;
        for (int ss = ss0; ss < ss1; ++ss) mine += (tot[(ss + a.n_mu) % n_seg] + 1) & ~1;
        int incl = mine;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        int pos = incl - mine;
        for (int ss = ss0; ss < ss1; ++ss) {
            const int s = (ss + a.n_mu) % n_seg;
            // packed back to back (fp32 kernel: jobs carry their own positions), or - seg_cap > 0 - one fixed slot of
            // seg_cap entries per segment, the layout the generic-precision kernel reads with seg_count
            base[s] = a.seg_cap > 0 ? s * a.seg_cap : pos;
            pos += (tot[s] + 1) & ~1;
            if (a.seg_cap > 0 && tot[s] + 1 > a.seg_cap) a.counters->overflow = 1;
        }
        if (lane == 31 && a.seg_cap == 0 && incl > a.pool_cap) a.counters->overflow = 1;
    }
    __syncthreads();
    for (int s = tid; s < n_seg; s += kPrepThreads) off[s] += base[s];
    __syncthreads();
    // ---- pass 2: write the entries; cntc[s][column] is the running position inside this CTA's block ------------
    for (int j = c0 + warp; j < c0 + cols; j += n_warps) {
        int *col = cntc + (j - c0);
        walk_column(a, reg, j, lane, s_cand[warp], [&](size_t c, int b, int t, double m, double wc) {
            const unsigned same0 = __match_any_sync(0xffffffffu, t != 0 ? b : -1);
            const unsigned same = __match_any_sync(0xffffffffu, t != 0 ? b * 4 + t : -1);
            int p0 = 0, pt = 0;
            if (t != 0) {  // rank among the chunk's cells of this mu-bin / of this (mu-bin, type), in row order
                p0 = off[b] + col[(size_t)b * cc] + __popc(same0 & ((1u << lane) - 1u));
                pt = off[t * a.n_mu + b] + col[(size_t)(t * a.n_mu + b) * cc] + __popc(same & ((1u << lane) - 1u));
            }
            __syncwarp();
            if (t != 0 && lane == __ffs(same0) - 1) col[(size_t)b * cc] += __popc(same0);
            if (t != 0 && lane == __ffs(same) - 1) col[(size_t)(t * a.n_mu + b) * cc] += __popc(same);
            __syncwarp();
            if (t != 0 && p0 < a.pool_cap && pt < a.pool_cap) {
                const double ac = doppler_minus_one(a.vel[c], a.mode);
                const double wl = wc * (a.lb.c[t][0] + a.lb.c[t][1] * m + a.lb.c[t][2] * m * m);
                EntT e;
                e.x = (decltype(e.x))ac;
                e.y = (decltype(e.y))(-wc);
                pool[p0] = e;
                e.y = (decltype(e.y))wl;
                pool[pt] = e;
            }
        });
    }
    if (rank != 0) return;
    // ---- rank 0 finalises the phase: pad odd segments, job list (contrast-carrying kinds 1, 2 first) -------------
    for (int s = tid; s < n_seg; s += kPrepThreads) {
        const int c = tot[s];
        if ((c & 1) && base[s] + c < a.pool_cap) {
            EntT z;
            z.x = 0;
            z.y = 0;
            pool[base[s] + c] = z;
        }
        if (a.seg_count) a.seg_count[p * n_seg + s] = c;
    }
    if (warp == 0) {
        const int per_lane = (n_seg + 31) / 32;
        const int ss0 = min(n_seg, lane * per_lane), ss1 = min(n_seg, ss0 + per_lane);
        int nj = 0, wsum = 0;
        for (int ss = ss0; ss < ss1; ++ss) {
            const int c = tot[(ss + a.n_mu) % n_seg];
            nj += (c + kActiveJobCap - 1) / kActiveJobCap;
            wsum += c;
        }
        int incl = nj;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        int k = incl - nj;
        for (int ss = ss0; ss < ss1; ++ss) {
            const int s = (ss + a.n_mu) % n_seg;
            const int c = tot[s];
            for (int o = 0; o < c; o += kActiveJobCap) {
                ActiveJob jb;
                jb.begin = p * a.pool_cap + base[s] + o;  // fits: host checks n_phases * pool_cap < 2^31
                jb.count = min(kActiveJobCap, c - o);
                jb.kind = s / a.n_mu;
                jb.row = s - jb.kind * a.n_mu;
                if (k < a.job_cap) a.jobs[(size_t)p * a.job_cap + k] = jb;
                ++k;
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) wsum += __shfl_xor_sync(0xffffffffu, wsum, d);
        const int n_jobs_total = __shfl_sync(0xffffffffu, incl, 31);
        if (lane == 0) {
            a.n_jobs[p] = min(n_jobs_total, a.job_cap);
            a.work[p] = wsum;
            a.n_active[p] = covered;
        }
    }
}

}  // namespace soap
