// a3 + a5 + a6 of SURVEY section 8 for fp32 spectra: the warp-specialised shift-interpolate-accumulate
// kernel (direct form).
//
//   out[m] = sum over entries e of  W_e * lerp(S_row(e); m + delta_e(m)),   delta_e(m) = a_e (lambda0/k + m)
//
// (Alg. 1 / Eq. 3 with Eq. 5-9 written as a gather; see sia.cuh for the
// generic-precision kernel that serves fp64 I/O.)  An entry is a (column, mu-bin) pair with its binned
// weight, or a single cell; entries of a spectrum row are ordered by shift factor a_e.
//
// The path is bound by FP32 instruction issue: one issue slot per SM sub-partition
// per clock, and the 3 FMAs of a lerp-accumulate are the only instructions the method needs per
// (entry, pixel).  Everything here exists to keep every other instruction out of the consumers' loop:
//
//   * CTA = 4 consumer warps + 1 producer warp.  A consumer thread owns R = 16 pixels of a 2048-pixel
//     wavelength tile (pixel m_t0 + tid + 128 r: conflict-free shared-memory reads, coalesced stores).
//   * "jobs" = (spectrum row, <= 128 entries).  The producer warp keeps a ring of kStages jobs in flight:
//     lane 0 issues two 1-D TMA bulk copies per job (the span of the row the tile's shifts can reach, and
//     the job's raw entries), then the whole warp turns the raw entries into what the consumers need:
//       - record {W a, -W q, W, 128 W a} per entry, so that a consumer forms W t for its first pixel with ONE
//         FMA (W a (lambda0/k + m) - W q) and for pixel r with one more (+ 128 W a r): no floor, no test;
//       - a run table: maximal groups of consecutive entries whose integer shift q is the same for every
//         pixel of the tile.  Consumers load their 16 samples and 16 sample differences once per run.
//       - entries whose q changes inside the tile ("flips", ~1 %) become runs of their own and take a
//         per-pixel path.  The producer also writes the clamp-to-edge halo (reading S8) of end tiles.
//     Full/empty mbarriers per stage; consumers never meet a CTA-wide barrier.
//   * per (entry, thread): 1 LDS.128 (broadcast) + 1 FFMA + 24 packed FFMA2 (fma.rn.f32x2: two pixels per
//     issue slot, so the FP32 pipe and not instruction issue is the limit) for 16 pixels.  Measured on
//     B200: FFMA2 runs at the full lane rate (126 of 128 lane-FMA/clk/SM) only with one scalar-broadcast
//     operand; with three register-pair operands it drops to ~70.  Hence W t_r d_r is split as
//     (W t_0) d_r + (128 W a) (r d_r) with r d_r kept in registers per run.
//   * precision: only the shift delta (|delta| < ~50) is formed in fp32, never the absolute source
//     coordinate; fp32 partial sums are folded into fp64 every kFold entries.
//   * quiet launch: the flattened (tile, entry) work list is cut into equal contiguous ranges, one per
//     CTA, grid = resident CTA slots (one wave, no tail); a CTA writes one fp64 partial per tile it
//     touches and reduce_ranges_kernel adds the partials of a tile in CTA order (deterministic).
//   * active launch: CTA = (tile, phase); the post-shift contrast (I_ratio of Eq. 3) multiplies each
//     kind's fp64 sum once per pixel (a6).
#pragma once
#include <climits>
#include <cstdint>
#include <cuda_runtime.h>

#include "ptx_helpers.cuh"

namespace soap {
namespace f32 {

constexpr int kConsumerWarps = 4;
constexpr int kConsumers = 32 * kConsumerWarps;  // consumer threads
constexpr int kThreads = kConsumers + 32;         // + producer warp
constexpr int kR = 16;                            // pixels per consumer thread
constexpr int kTile = kConsumers * kR;            // pixels per tile
constexpr int kStages = 4;                        // jobs in flight
constexpr int kJobCap = 128;                      // entries per job (even)
constexpr int kFold = 64;                         // fp32 -> fp64 fold interval (entries)
constexpr int kMaxSeg = 3 * 64;                   // 3 kinds x SOAP_MAX_MU
constexpr int kFlip = INT_MIN;                    // run marker: per-pixel path

struct Params {
    const float *base[3];      // spectrum tables per kind (quiet launch: base[0] only)
    const float *contrast[3];  // per-pixel multiplier per kind or nullptr (== 1); kind 0 unused
    long long pitch, n_pix;
    double c0;                 // lambda0 / dlambda
    int n_mu;
    int halo;                  // H: multiple of 4, >= max |delta| + 2
    const float2 *ent;         // raw entries (a_e, W_e)
    // quiet launch
    const int *row_start;      // [n_mu + 1] entry offsets (even)
    int n_tiles;
    double *partial;           // [gridDim.x][max_seg][kTile]
    int max_seg;
    // active launch
    const int *seg_count;      // [n_phases][3][n_mu]
    int seg_cap;               // entries reserved per segment (even)
    float *out;                // [n_phases][out_pitch]
    long long out_pitch;
};

// First unit of CTA c when U units (U even) are cut into G contiguous ranges with even boundaries.
__host__ __device__ inline long long range_begin(long long c, long long U, long long G) {
    return 2 * ((c * (U / 2)) / G);
}

__host__ __device__ constexpr int span_px(int halo) { return kTile + 2 * halo + 4; }

struct StageLayout {
    size_t row_bytes, raw_off, rec_off, run_off, stage_bytes;
};
__host__ __device__ inline StageLayout stage_layout(int halo) {
    StageLayout l;
    l.row_bytes = ((size_t)span_px(halo) * sizeof(float) + 127) & ~(size_t)127;
    l.raw_off = l.row_bytes;
    l.rec_off = l.raw_off + kJobCap * sizeof(float2);
    l.run_off = l.rec_off + kJobCap * sizeof(float2);
    l.stage_bytes = (l.run_off + (kJobCap + 2) * sizeof(int2) + 127) & ~(size_t)127;
    return l;
}
constexpr size_t kHeaderBytes = 128 + 2 * kMaxSeg * sizeof(int);  // mbarriers + segment table (multiple of 128)
constexpr size_t kFinBytes = (size_t)kTile * sizeof(double);      // active launch: per-pixel fp64 delta accumulators
__host__ inline size_t smem_bytes(int halo, bool active) {
    return kHeaderBytes + (active ? kFinBytes : 0) + kStages * stage_layout(halo).stage_bytes;
}

struct Job {
    long long tile;
    int seg;    // segment index (kind * n_mu + row)
    int begin;  // first entry (global index, even)
    int count;  // entries, <= kJobCap
};

// Enumerates the jobs of a CTA: for each tile of its range, for each segment, chunks of <= kJobCap
// entries.  The producer (twice: issue and post-process) and every consumer walk the same sequence.
struct WorkIter {
    long long t, t_end, u0, u1, E;
    int s, pos, e_lo, e_hi;
    bool ranged;
    __device__ void open_tile() {
        if (ranged) {
            const long long lo = u0 - t * E, hi = u1 - t * E;
            e_lo = (int)(lo > 0 ? lo : 0);
            e_hi = (int)(hi < E ? hi : E);
        } else {
            e_lo = 0;
            e_hi = INT_MAX;
        }
        s = 0;
        pos = 0;
    }
    __device__ bool next(const int *seg_lo, const int *seg_hi, int n_seg, Job &j) {
        for (;;) {
            while (s < n_seg) {
                const int lo = max(seg_lo[s], e_lo), hi = min(seg_hi[s], e_hi);
                const int p = max(pos, lo);
                if (p < hi) {
                    j.tile = t;
                    j.seg = s;
                    j.begin = p;
                    j.count = min(hi - p, kJobCap);
                    pos = p + j.count;
                    return true;
                }
                ++s;
            }
            if (t >= t_end) return false;
            ++t;
            open_tile();
        }
    }
};

template <bool ACTIVE>
__global__ void __launch_bounds__(kThreads, 3) sia_f32_kernel(const Params p) {
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *bar_tma = reinterpret_cast<uint64_t *>(smem);  // [kStages] TMA landed      (count 1 + tx)
    uint64_t *bar_ready = bar_tma + kStages;                 // [kStages] records written (count 1)
    uint64_t *bar_empty = bar_ready + kStages;               // [kStages] consumers done  (count kConsumerWarps)
    int *seg_lo = reinterpret_cast<int *>(smem + 128);
    int *seg_hi = seg_lo + kMaxSeg;
    const int H = p.halo;
    const int span = span_px(H);
    const StageLayout L = stage_layout(H);
    double *fin = reinterpret_cast<double *>(smem + kHeaderBytes);  // active launch only: [kR][kConsumers]
    unsigned char *stage0 = smem + kHeaderBytes + (ACTIVE ? kFinBytes : 0);

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int n_seg = ACTIVE ? 3 * p.n_mu : p.n_mu;

    // ---- this CTA's work ---------------------------------------------------------------------------
    WorkIter w0;
    if (ACTIVE) {
        const int phase = blockIdx.y;
        for (int s = tid; s < n_seg; s += kThreads) {
            const int gs = phase * n_seg + s;
            seg_lo[s] = gs * p.seg_cap;  // fits: host checks n_phases*3*n_mu*seg_cap < 2^31
            seg_hi[s] = gs * p.seg_cap + p.seg_count[gs];
        }
        w0.ranged = false;
        w0.t = w0.t_end = blockIdx.x;
        w0.u0 = w0.u1 = w0.E = 0;
    } else {
        for (int s = tid; s < n_seg; s += kThreads) {
            seg_lo[s] = p.row_start[s];
            seg_hi[s] = p.row_start[s + 1];
        }
        const long long E = p.row_start[p.n_mu];
        const long long U = E * p.n_tiles;
        w0.ranged = true;
        w0.E = E;
        w0.u0 = range_begin(blockIdx.x, U, gridDim.x);
        w0.u1 = range_begin(blockIdx.x + 1, U, gridDim.x);
        if (w0.u1 <= w0.u0) return;  // more CTAs than work (whole CTA leaves before any barrier)
        w0.t = w0.u0 / E;
        w0.t_end = (w0.u1 - 1) / E;
    }
    w0.open_tile();
    const long long t_first = w0.t, t_last = w0.t_end;
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&bar_tma[s], 1);
            mbar_init(&bar_ready[s], 1);
            mbar_init(&bar_empty[s], kConsumerWarps);
        }
        fence_mbar_init();
    }
    __syncthreads();

    if (warp == kConsumerWarps) {
        // =============================== producer warp ===============================================
        WorkIter it_issue = w0, it_proc = w0;
        Job ji, jp;
        bool have_ji = false, more = true;
        int n_issued = 0, n_proc = 0;
        for (;;) {
            // -- keep the TMA ring full -----------------------------------------------------------------
            for (;;) {
                if (!have_ji && more) {
                    more = it_issue.next(seg_lo, seg_hi, n_seg, ji);
                    have_ji = more;
                }
                if (!have_ji || n_issued >= n_proc + kStages) break;
                const int st = n_issued % kStages;
                const uint32_t par = (uint32_t)(((n_issued / kStages) & 1) ^ 1);
                int free_ = 0;
                if (lane == 0) free_ = mbar_try_wait(&bar_empty[st], par) ? 1 : 0;
                free_ = __shfl_sync(0xffffffffu, free_, 0);
                if (!free_) break;
                if (lane == 0) {
                    const long long s_start = ji.tile * kTile - H;  // global pixel of smem position 0 (multiple of 4)
                    const long long g_lo = s_start < 0 ? 0 : s_start;
                    const long long g_hi = (s_start + span) < p.pitch ? (s_start + span) : p.pitch;
                    const uint32_t row_bytes = (uint32_t)((g_hi - g_lo) * (long long)sizeof(float));
                    const int kind = ACTIVE ? ji.seg / p.n_mu : 0;
                    const int row = ACTIVE ? ji.seg - kind * p.n_mu : ji.seg;
                    const float *src = p.base[kind] + (long long)row * p.pitch + g_lo;
                    const uint32_t ent_bytes = (uint32_t)(((ji.count + 1) & ~1) * (int)sizeof(float2));
                    unsigned char *sb = stage0 + (size_t)st * L.stage_bytes;
                    fence_proxy_async_smem();
                    mbar_arrive_expect_tx(&bar_tma[st], row_bytes + ent_bytes);
                    tma_load_1d(sb + (size_t)(g_lo - s_start) * sizeof(float), src, row_bytes, &bar_tma[st]);
                    tma_load_1d(sb + L.raw_off, p.ent + ji.begin, ent_bytes, &bar_tma[st]);
                }
                ++n_issued;
                have_ji = false;
            }
            if (n_proc < n_issued) {
                // -- post-process one landed job: records, run table, edge halo ---------------------------
                it_proc.next(seg_lo, seg_hi, n_seg, jp);
                const int st = n_proc % kStages;
                mbar_wait(&bar_tma[st], (uint32_t)((n_proc / kStages) & 1));
                unsigned char *sb = stage0 + (size_t)st * L.stage_bytes;
                float *rs = reinterpret_cast<float *>(sb);
                const float2 *raw = reinterpret_cast<const float2 *>(sb + L.raw_off);
                float2 *rec = reinterpret_cast<float2 *>(sb + L.rec_off);
                int2 *runs = reinterpret_cast<int2 *>(sb + L.run_off);
                const long long m_t0 = jp.tile * kTile;
                const float c_first = (float)(p.c0 + (double)m_t0);
                const float c_last = (float)(p.c0 + (double)(m_t0 + kTile - 1));
                int n_runs = 0, carry = kFlip;  // kFlip never equals a q: the first entry opens a run
                for (int i0 = 0; i0 < jp.count; i0 += 32) {
                    const int i = i0 + lane;
                    const bool valid = i < jp.count;
                    int code = kFlip;
                    if (valid) {
                        const float2 en = raw[i];
                        const float qf = floorf(en.x * c_first), ql = floorf(en.x * c_last);
                        int qi = (int)qf;
                        qi = max(-H, min(H + 2, qi));
                        rec[i] = make_float2(en.y, en.y * en.x);  // {W, W a}
                        if (qf == ql) code = qi;
                    }
                    int prev = __shfl_up_sync(0xffffffffu, code, 1);
                    if (lane == 0) prev = carry;
                    const bool start = valid && (code == kFlip || code != prev);
                    const unsigned mask = __ballot_sync(0xffffffffu, start);
                    if (start) runs[1 + n_runs + __popc(mask & ((1u << lane) - 1u))] = make_int2(i, code);
                    n_runs += __popc(mask);
                    carry = __shfl_sync(0xffffffffu, code, 31);
                }
                if (lane == 0) {
                    runs[0] = make_int2(n_runs, 0);
                    runs[1 + n_runs] = make_int2(jp.count, 0);  // sentinel: end of the last run
                }
                const long long s_start = m_t0 - H;
                if (s_start < 0) {  // clamp-to-edge below the grid (reading S8)
                    const int n = (int)(-s_start);
                    const float v = rs[n];
                    for (int q = lane; q < n; q += 32) rs[q] = v;
                }
                if (s_start + span > p.n_pix) {  // ... and above it
                    const int first = (int)(p.n_pix - s_start);
                    const float v = rs[first - 1];
                    for (int q = first + lane; q < span; q += 32) rs[q] = v;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&bar_ready[st]);
                ++n_proc;
            } else if (!have_ji) {
                break;  // everything issued and processed
            } else {
                // ring full of jobs the consumers still hold: wait for the oldest stage
                const int st = n_issued % kStages;
                mbar_wait(&bar_empty[st], (uint32_t)(((n_issued / kStages) & 1) ^ 1));
            }
        }
        return;
    }

    // =================================== consumer warps ===============================================
    WorkIter it = w0;
    Job job;
    bool have = it.next(seg_lo, seg_hi, n_seg, job);
    int n_done = 0;
    const int base0 = H + tid;  // smem position of pixel r = 0 at zero shift
    for (long long tile = t_first; tile <= t_last; ++tile) {
        const long long m_t0 = tile * kTile;
        const float cmf = (float)(p.c0 + (double)(m_t0 + tid));  // lambda0/k + m of this thread's first pixel
        float2 acc[kR / 2];  // pair k = pixels r = 2k, 2k + 1: the operands of one packed FMA
        double tot[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            if (r & 1) acc[r / 2].y = 0.f;
            else acc[r / 2].x = 0.f;
            tot[r] = 0.0;
            if (ACTIVE) fin[r * kConsumers + tid] = 0.0;  // only this thread ever touches its 16 slots
        }
        int cnt = 0, cur_kind = 0;
        auto fold = [&]() {
#pragma unroll
            for (int k = 0; k < kR / 2; ++k) {
                tot[2 * k] += (double)acc[k].x;
                tot[2 * k + 1] += (double)acc[k].y;
                acc[k] = make_float2(0.f, 0.f);
            }
            cnt = 0;
        };
        auto fold_kind = [&](int kind) {  // a6: post-shift contrast (I_ratio of Eq. 3) per output pixel
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const long long m = m_t0 + tid + kConsumers * r;
                double c = 1.0;
                if (kind > 0 && p.contrast[kind] != nullptr && m < p.n_pix) c = (double)p.contrast[kind][m];
                if (ACTIVE) fin[r * kConsumers + tid] += c * tot[r];
                tot[r] = 0.0;
            }
        };

        while (have && job.tile == tile) {
            const int st = n_done % kStages;
            mbar_wait(&bar_ready[st], (uint32_t)((n_done / kStages) & 1));
            const unsigned char *sb = stage0 + (size_t)st * L.stage_bytes;
            const float *rs = reinterpret_cast<const float *>(sb);
            const float2 *raw = reinterpret_cast<const float2 *>(sb + L.raw_off);
            const float2 *rec = reinterpret_cast<const float2 *>(sb + L.rec_off);
            const int2 *runs = reinterpret_cast<const int2 *>(sb + L.run_off);
            if (ACTIVE) {
                const int kind = job.seg / p.n_mu;
                if (kind != cur_kind) {
                    fold();
                    fold_kind(cur_kind);
                    cur_kind = kind;
                }
            }
            const int n_runs = runs[0].x;
            for (int ri = 1; ri <= n_runs; ++ri) {
                const int2 run = runs[ri];
                const int nxt = runs[ri + 1].x;
                if (run.y == kFlip) {
                    // integer shift changes inside the tile: per-pixel floor
                    const float2 en = raw[run.x];
#pragma unroll
                    for (int r = 0; r < kR; ++r) {
                        const float cm = cmf + (float)(kConsumers * r);
                        const float q = floorf(en.x * cm);
                        const float t = fmaf(en.x, cm, -q);
                        int qi = (int)q;
                        qi = max(-H, min(H + 2, qi));
                        const float s0 = rs[base0 + kConsumers * r + qi], s1 = rs[base0 + kConsumers * r + qi + 1];
                        float &ar = (r & 1) ? acc[r / 2].y : acc[r / 2].x;
                        ar = fmaf(en.y, fmaf(t, s1 - s0, s0), ar);
                    }
                    if (++cnt >= kFold) fold();
                    continue;
                }
                // With t = a c - q (c = lambda0/k + m, q the run's integer shift), W lerp = W (s + t d) regroups
                // to W u + (W a) v with u = s - q d and v = c d: u_r, v_r are per-pixel registers of the run and
                // every entry costs two FMAs per pixel, each with one scalar (broadcast) operand.
                float2 u[kR / 2], v[kR / 2];
                {
                    const float *wv = rs + base0 + run.y;
                    const float2 nq = bcast2(-(float)run.y);
#pragma unroll
                    for (int k = 0; k < kR / 2; ++k) {
                        const float2 s0 = make_float2(wv[kConsumers * 2 * k], wv[kConsumers * (2 * k + 1)]);
                        const float2 s1 = make_float2(wv[kConsumers * 2 * k + 1], wv[kConsumers * (2 * k + 1) + 1]);
                        const float2 d = fma2(bcast2(-1.f), s0, s1);
                        const float2 c = make_float2(cmf + (float)(kConsumers * 2 * k), cmf + (float)(kConsumers * (2 * k + 1)));
                        u[k] = fma2(nq, d, s0);
                        v[k] = fma2(c, d, bcast2(0.f));
                    }
                }
                int e = run.x;
                while (e < nxt) {
                    const int n = min(nxt - e, kFold - cnt);
#pragma unroll 2
                    for (int i = 0; i < n; ++i) {
                        const float2 rc = rec[e + i];  // {W, W a}
#pragma unroll
                        for (int k = 0; k < kR / 2; ++k) acc[k] = fma2(bcast2(rc.x), u[k], acc[k]);  // (1) + W u_r
#pragma unroll
                        for (int k = 0; k < kR / 2; ++k) acc[k] = fma2(bcast2(rc.y), v[k], acc[k]);  // (2) + W a v_r
                    }
                    e += n;
                    cnt += n;
                    if (cnt >= kFold) fold();
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_empty[st]);
            ++n_done;
            have = it.next(seg_lo, seg_hi, n_seg, job);
        }

        // ---- store ---------------------------------------------------------------------------------
        fold();
        if (ACTIVE) {
            fold_kind(cur_kind);
            float *o = p.out + (long long)blockIdx.y * p.out_pitch;
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const long long m = m_t0 + tid + kConsumers * r;
                if (m < p.n_pix) o[m] = (float)fin[r * kConsumers + tid];
            }
        } else {
            double *o = p.partial + ((long long)blockIdx.x * p.max_seg + (tile - t_first)) * kTile;
#pragma unroll
            for (int r = 0; r < kR; ++r) o[tid + kConsumers * r] = tot[r];
        }
    }
}

// a6 for the quiet spectrum: adds, in CTA order, the partials of every CTA whose range touched the
// pixel's tile, and rounds once to fp32.  blockDim.x divides kTile, so a block lies inside one tile and
// thread 0 finds the contributing CTAs once for the block.
constexpr int kReduceThreads = 256;
constexpr int kReduceMaxSrc = 64;
__global__ void __launch_bounds__(kReduceThreads)
reduce_ranges_kernel(const double *__restrict__ partial, int max_seg, const int *__restrict__ row_start, int n_mu,
                     int n_cta, int n_tiles, long long n_pix, float *__restrict__ out) {
    __shared__ long long s_src[kReduceMaxSrc];  // element offset of each contributing partial tile
    __shared__ int s_n, s_c0, s_c1;
    const long long m0 = (long long)blockIdx.x * kReduceThreads;
    const long long t = m0 / kTile;
    const long long E = row_start[n_mu], U = E * n_tiles, G = n_cta;
    if (threadIdx.x == 0) {
        int n = 0;
        s_c0 = 0;
        s_c1 = 0;
        if (U > 0) {
            const long long ub = t * E, ue = ub + E;
            long long c = (ub * G) / U;
            while (c > 0 && range_begin(c, U, G) > ub) --c;
            while (c + 1 < G && range_begin(c + 1, U, G) <= ub) ++c;
            s_c0 = (int)c;
            for (; c < G; ++c) {
                const long long b = range_begin(c, U, G), e = range_begin(c + 1, U, G);
                if (b >= ue) break;
                if (e <= b || e <= ub) continue;
                if (n < kReduceMaxSrc) s_src[n] = (c * max_seg + (t - b / E)) * kTile;
                ++n;
            }
            s_c1 = (int)c;
        }
        s_n = n;
    }
    __syncthreads();
    const long long m = m0 + threadIdx.x;
    if (m >= n_pix) return;
    const long long off = m - t * kTile;
    double v = 0.0;
    if (s_n <= kReduceMaxSrc) {
        for (int k = 0; k < s_n; ++k) v += partial[s_src[k] + off];
    } else {  // more contributing CTAs than the table holds (tiny entry lists): walk the ranges directly
        const long long ub = t * E;
        for (long long c = s_c0; c < s_c1; ++c) {
            const long long b = range_begin(c, U, G), e = range_begin(c + 1, U, G);
            if (e <= b || e <= ub) continue;
            v += partial[(c * max_seg + (t - b / E)) * kTile + off];
        }
    }
    out[m] = (float)v;
}

}  // namespace f32
}  // namespace soap
