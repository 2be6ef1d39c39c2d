// a3 + a5 + a6 of SURVEY section 8: the shift-interpolate-accumulate kernel (direct form).
//
//   out[m] = sum over entries e of  W_e * lerp(S_row(e); m + delta_e(m)),   delta_e(m) = a_e (lambda0/k + m)
//
// which is Alg. 1 / Eq. 3 of the paper with Eq. 5-9 written as a gather:
// a_e = D_e - 1 is the entry's Doppler shift factor, so m + delta_e(m) = (lambda_m D_e - lambda_0)/k is
// the source coordinate of output pixel m; its integer part q and fraction t are closed-form, no search.
// An entry is a (column, mu-bin) pair with its binned weight (pre-binned form) or a single cell.
// This generic-precision kernel serves fp64 I/O (config C1); fp32 spectra take the warp-specialised kernel of
// sia_f32.cuh, the one bench.py measures.
//
// Mapping to the SM (sm_100a):
//   * one CTA = one wavelength tile of kThreads*R pixels x one chunk of the entry list (quiet) or one
//     phase (active).  Thread t owns pixels m_t0 + t + kThreads*r, r < R (interleaved: conflict-free
//     shared-memory reads, coalesced stores).
//   * "jobs" = (spectrum row, <= kEntCap entries).  For every job one elected thread issues two TMA bulk
//     copies (cp.async.bulk -> UBLKCP): the span of the row this tile's shifts can reach, and the job's
//     entries; an mbarrier ring of kStages stages keeps kStages-1 jobs in flight behind the math.
//   * inner loop: entries of a row are ordered by shift factor, so consecutive entries share the integer
//     shift q.  The thread keeps the R samples S[m_r+q] and differences S[m_r+q+1]-S[m_r+q] of its pixels
//     in registers and reloads them from shared memory only when q changes; per (entry, pixel) that
//     leaves exactly the 3 FP32 FMAs of a lerp-accumulate:  t_r = t_0 + (a*kThreads) r  (1),
//     acc += W s_r (2), acc += (W t_r) d_r (3) - no shared-memory traffic, no index arithmetic.
//     An entry whose q differs across the thread's pixels (a "flip", < 1 % of entries) takes a generic
//     per-pixel path.
//   * precision: only the *shift* delta (|delta| < ~50) is formed in fp32, never the absolute source
//     coordinate (~7e5), and fp32 partial sums are folded into fp64 accumulators every <= 64 entries and
//     at every window change; the 1 cm/s line-RV budget of north_star needs both.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "ptx_helpers.cuh"

namespace soap {

constexpr int kThreads = 128;   // threads per CTA
constexpr int kStages = 3;      // TMA ring depth
constexpr int kEntCap = 256;    // entries per job
constexpr int kFlushEvery = 64; // fp32 -> fp64 fold interval (entries)
constexpr int kMaxSeg = 3 * 64; // 3 kinds x SOAP_MAX_MU

template <typename T> struct SiaTraits;
template <> struct SiaTraits<float> {
    static constexpr int R = 8;
    using Ent = float2;
};
template <> struct SiaTraits<double> {
    static constexpr int R = 4;
    using Ent = double2;
};

template <typename T>
struct SiaParams {
    const T *base[3];       // spectrum tables per kind (quiet kernel: base[0] only)
    const T *contrast[3];   // per-pixel multiplier per kind or nullptr (== 1); kind 0 unused
    long long pitch, n_pix;
    double c0;              // lambda0 / dlambda
    int n_mu;
    int halo;               // H: multiple of 4, >= max |delta| + 2
    const typename SiaTraits<T>::Ent *ent;
    const int *row_start;   // quiet: [n_mu + 1] entry offsets (even)
    const int *seg_count;   // active: [n_phases][3][n_mu]
    int seg_cap;            // active: entries reserved per segment
    int n_splits;           // quiet: number of entry chunks (gridDim.y)
    double *partial;        // quiet: [n_splits][part_pitch]
    long long part_pitch;
    T *out;                 // active: [n_phases][out_pitch]
    long long out_pitch;
};

template <typename T>
__host__ __device__ constexpr int sia_tile_px() {
    return kThreads * SiaTraits<T>::R;
}

template <typename T>
__host__ inline size_t sia_smem_bytes(int halo) {
    const size_t span = (size_t)sia_tile_px<T>() + 2 * (size_t)halo + 4;
    size_t b = 128;                                               // mbarriers
    b += 2 * kMaxSeg * sizeof(int);                               // segment tables
    b = (b + 127) & ~(size_t)127;
    b += kStages * ((span * sizeof(T) + 127) & ~(size_t)127);     // row spans
    b += kStages * kEntCap * sizeof(typename SiaTraits<T>::Ent);  // entries
    return b;
}

struct Job {
    int seg;    // segment index (kind * n_mu + row)
    int begin;  // first entry (global index, even)
    int count;  // entries in this job, <= kEntCap
};

// Walks the segment table; identical sequence for the producer thread and for the consumers.
struct JobIter {
    const int *seg_begin, *seg_count;
    int n_seg, seg, off;
    __device__ JobIter(const int *b, const int *c, int n) : seg_begin(b), seg_count(c), n_seg(n), seg(0), off(0) {}
    __device__ bool next(Job &j) {
        while (seg < n_seg && off >= seg_count[seg]) {
            ++seg;
            off = 0;
        }
        if (seg >= n_seg) return false;
        const int left = seg_count[seg] - off;
        j.seg = seg;
        j.begin = seg_begin[seg] + off;
        j.count = left < kEntCap ? left : kEntCap;
        off += kEntCap;
        return true;
    }
};

template <typename T>
__device__ __forceinline__ T fma_t(T a, T b, T c);
template <>
__device__ __forceinline__ float fma_t<float>(float a, float b, float c) {
    return fmaf(a, b, c);
}
template <>
__device__ __forceinline__ double fma_t<double>(double a, double b, double c) {
    return fma(a, b, c);
}

template <typename T, bool ACTIVE>
__global__ void __launch_bounds__(kThreads) sia_kernel(const SiaParams<T> p) {
    constexpr int R = SiaTraits<T>::R;
    constexpr int TP = kThreads * R;
    using Ent = typename SiaTraits<T>::Ent;

    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smem);
    int *seg_begin = reinterpret_cast<int *>(smem + 128);
    int *seg_count = seg_begin + kMaxSeg;
    const int H = p.halo;
    const int span = TP + 2 * H + 4;
    const size_t row_stride = ((size_t)span * sizeof(T) + 127) & ~(size_t)127;
    unsigned char *rows0 = smem + ((128 + 2 * kMaxSeg * sizeof(int) + 127) & ~(size_t)127);
    unsigned char *ents0 = rows0 + kStages * row_stride;

    const int tid = threadIdx.x;
    const long long m_t0 = (long long)blockIdx.x * TP;
    const long long s_start = m_t0 - H;  // global pixel index of smem position 0 (multiple of 4)
    const int n_seg = ACTIVE ? 3 * p.n_mu : p.n_mu;

    // ---- segment table -------------------------------------------------------------------------
    if (ACTIVE) {
        const int phase = blockIdx.y;
        for (int s = tid; s < n_seg; s += kThreads) {
            const int gs = phase * n_seg + s;
            seg_begin[s] = gs * p.seg_cap;  // fits: host checks n_phases*3*n_mu*seg_cap < 2^31
            seg_count[s] = p.seg_count[gs];
        }
    } else {
        const int E = p.row_start[p.n_mu];
        const int cs = (((E + p.n_splits - 1) / p.n_splits) + 1) & ~1;  // even chunk size
        const int e_lo = blockIdx.y * cs;
        const int e_hi = min(E, e_lo + cs);
        for (int s = tid; s < n_seg; s += kThreads) {
            const int b = max(p.row_start[s], e_lo);
            const int e = min(p.row_start[s + 1], e_hi);
            seg_begin[s] = b;
            seg_count[s] = max(0, e - b);
        }
    }
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&mbar[s], 1);
        fence_mbar_init();
    }
    __syncthreads();

    // ---- what part of a row this tile stages -----------------------------------------------------
    const long long g_lo = s_start < 0 ? 0 : s_start;
    const long long g_hi = (s_start + span) < p.pitch ? (s_start + span) : p.pitch;
    const uint32_t row_bytes = (uint32_t)((g_hi - g_lo) * (long long)sizeof(T));
    const int dst_off = (int)(g_lo - s_start);
    const bool patch_left = s_start < 0;
    const bool patch_right = (s_start + span) > p.n_pix;

    auto issue = [&](const Job &j, int st) {
        const int kind = ACTIVE ? j.seg / p.n_mu : 0;
        const int row = ACTIVE ? j.seg - kind * p.n_mu : j.seg;
        const T *src = p.base[kind] + (long long)row * p.pitch + g_lo;
        const uint32_t ent_bytes = (uint32_t)(((j.count + 1) & ~1) * (int)sizeof(Ent));
        mbar_arrive_expect_tx(&mbar[st], row_bytes + ent_bytes);
        tma_load_1d(rows0 + st * row_stride + (size_t)dst_off * sizeof(T), src, row_bytes, &mbar[st]);
        tma_load_1d(ents0 + (size_t)st * kEntCap * sizeof(Ent), p.ent + j.begin, ent_bytes, &mbar[st]);
    };

    // ---- per-thread pixel state ------------------------------------------------------------------
    const int base0 = H + tid;  // smem position of pixel r = 0 at zero shift
    const T cmf = (T)(p.c0 + (double)(m_t0 + tid));                       // lambda0/k + m, first pixel
    const T cml = (T)(p.c0 + (double)(m_t0 + tid + kThreads * (R - 1)));  // ... last pixel
    T acc[R], s[R], d[R];
    double tot[R], fin[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        acc[r] = (T)0;
        s[r] = (T)0;
        d[r] = (T)0;
        tot[r] = 0.0;
        fin[r] = 0.0;
    }
    T curq = (T)1e30;  // forces a window load at the first entry of a job
    int cur_kind = 0;

    auto flush = [&]() {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            tot[r] += (double)acc[r];
            acc[r] = (T)0;
        }
    };
    auto fold_kind = [&](int kind) {  // a6: post-shift contrast (I_ratio of Eq. 3) applied per output pixel
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long m = m_t0 + tid + kThreads * r;
            double c = 1.0;
            if (kind > 0 && p.contrast[kind] != nullptr && m < p.n_pix) c = (double)p.contrast[kind][m];
            fin[r] += c * tot[r];
            tot[r] = 0.0;
        }
    };

    // ---- pipeline ----------------------------------------------------------------------------------
    JobIter prod(seg_begin, seg_count, n_seg), cons(seg_begin, seg_count, n_seg);
    int issued = 0, consumed = 0;
    if (tid == 0) {
        Job j;
        for (int i = 0; i < kStages - 1; ++i)
            if (prod.next(j)) {
                issue(j, issued % kStages);
                ++issued;
            }
    }
    Job job;
    while (cons.next(job)) {
        const int st = consumed % kStages;
        const uint32_t parity = (uint32_t)((consumed / kStages) & 1);
        __syncthreads();  // every thread is done with job consumed-1: its stage may be refilled
        if (tid == 0) {
            Job j;
            if (prod.next(j)) {
                issue(j, issued % kStages);
                ++issued;
            }
        }
        mbar_wait(&mbar[st], parity);
        T *rs = reinterpret_cast<T *>(rows0 + st * row_stride);
        const Ent *ents = reinterpret_cast<const Ent *>(ents0 + (size_t)st * kEntCap * sizeof(Ent));
        if (patch_left || patch_right) {  // clamp-to-edge outside the grid (reading S8)
            if (patch_left) {
                const int n = (int)(-s_start);
                const T v = rs[n];
                for (int q = tid; q < n; q += kThreads) rs[q] = v;
            }
            if (patch_right) {
                const int first = (int)(p.n_pix - s_start);
                const T v = rs[first - 1];
                for (int q = first + tid; q < span; q += kThreads) rs[q] = v;
            }
            __syncthreads();
        }
        if (ACTIVE) {
            const int kind = job.seg / p.n_mu;
            if (kind != cur_kind) {
                fold_kind(cur_kind);
                cur_kind = kind;
            }
        }
        curq = (T)1e30;
        for (int e0 = 0; e0 < job.count; e0 += kFlushEvery) {
            const int e1 = min(job.count, e0 + kFlushEvery);
            for (int e = e0; e < e1; ++e) {
                const Ent en = ents[e];
                const T a = en.x, W = en.y;
                T t0 = fma_t<T>(a, cmf, -curq);
                const T tl = fma_t<T>(a, cml, -curq);
                if (!(fmin(t0, tl) >= (T)0 && fmax(t0, tl) < (T)1)) {
                    const T q0 = floor(a * cmf), ql = floor(a * cml);
                    if (q0 != ql) {
                        // integer shift changes inside this thread's pixel set: generic per-pixel path
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const T cm = cmf + (T)(kThreads * r);
                            const T q = floor(a * cm);
                            const T t = fma_t<T>(a, cm, -q);
                            int qi = (int)q;
                            qi = max(-H, min(H + 2, qi));
                            const T s0 = rs[base0 + kThreads * r + qi], s1 = rs[base0 + kThreads * r + qi + 1];
                            acc[r] = fma_t<T>(W, fma_t<T>(t, s1 - s0, s0), acc[r]);
                        }
                        continue;
                    }
                    flush();
                    curq = q0;
                    int qi = (int)q0;
                    qi = max(-H, min(H + 2, qi));
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const T s0 = rs[base0 + kThreads * r + qi], s1 = rs[base0 + kThreads * r + qi + 1];
                        s[r] = s0;
                        d[r] = s1 - s0;
                    }
                    t0 = fma_t<T>(a, cmf, -curq);
                }
                const T wa = W * t0, wb = W * a;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    acc[r] = fma_t<T>(W, s[r], acc[r]);
                    acc[r] = fma_t<T>(fma_t<T>(wb, (T)(kThreads * r), wa), d[r], acc[r]);
                }
            }
            flush();
        }
        ++consumed;
    }

    // ---- store -------------------------------------------------------------------------------------
    if (ACTIVE) {
        fold_kind(cur_kind);
        T *o = p.out + (long long)blockIdx.y * p.out_pitch;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long m = m_t0 + tid + kThreads * r;
            if (m < p.n_pix) o[m] = (T)fin[r];
        }
    } else {
        double *o = p.partial + (long long)blockIdx.y * p.part_pitch;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long m = m_t0 + tid + kThreads * r;
            if (m < p.n_pix) o[m] = tot[r];
        }
    }
}

// a6 for the quiet spectrum: ordered sum of the entry-chunk partials (deterministic), cast to the
// output type; 4 pixels per thread, 128-bit stores when the output is fp32.
template <typename T>
__global__ void reduce_partials_kernel(const double *__restrict__ partial, long long part_pitch, int n_splits,
                                       long long n_pix, T *__restrict__ out) {
    const long long m0 = 4 * ((long long)blockIdx.x * blockDim.x + threadIdx.x);
    if (m0 >= n_pix) return;
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    if (m0 + 3 < n_pix) {
        for (int sidx = 0; sidx < n_splits; ++sidx) {
            const double2 *pp = reinterpret_cast<const double2 *>(partial + (long long)sidx * part_pitch + m0);
            const double2 x = pp[0], y = pp[1];
            v[0] += x.x;
            v[1] += x.y;
            v[2] += y.x;
            v[3] += y.y;
        }
        for (int k = 0; k < 4; ++k) out[m0 + k] = (T)v[k];
    } else {
        for (int k = 0; m0 + k < n_pix; ++k) {
            double a = 0.0;
            for (int sidx = 0; sidx < n_splits; ++sidx) a += partial[(long long)sidx * part_pitch + m0 + k];
            out[m0 + k] = (T)a;
        }
    }
}

}  // namespace soap
