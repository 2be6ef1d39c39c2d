// a3 of SURVEY section 8, composite-column form (SOAP_FORM_COMPOSITE) for fp32 spectra under solid-body rotation.
//
//   Q[m] = sum_j sum_b W[j,b] lerp(S_b; m + delta_j(m))  =  sum_j lerp(T_j; m + delta_j(m)),   T_j[n] = sum_b W[j,b] S_b[n]
//
// (Alg. 1 with Eq. 5-9 as a gather; cells pre-binned by (column, mu-bin) as BASELINE.json's
// north_star allows.)  Linear interpolation is linear in the spectrum and all cells of a column share one velocity, so
// the weighted rows of a column can be added BEFORE the shift: one FMA per (column, mu-bin, pixel) on unshifted
// samples, then one interpolation per (column, pixel) - instead of two FMAs per (column, mu-bin, pixel) plus a
// window set-up per run of entries.  Nothing depends on how the shifts are distributed, so fast rotators cost
// the same as slow ones ("composite-column form").
//
//   * A CTA of 512 threads holds a span of 2048 source pixels of EVERY mu-bin row in registers (thread i: pixels
//     n0 + i + 512 r of each row): 20 bins x 2048 px = 62 % of the SM's register file.  The span is an output tile of
//     L = 2048 - 2 H pixels plus the halo H the shifts can reach on either side.
//   * Columns are taken four at a time (a "quad" = two column pairs).  Compute phase: TU[r] = (T_j, T_j+1)[pixel r]
//     accumulates (W[j,b], W[j+1,b]) * S_b[r] with packed FFMA2 (the weight pair is half of an LDS.128-broadcast, the
//     sample a scalar-broadcast register): 4 FFMA2 per (pair, bin) per thread, straight-line per number of bins
//     present.  Column j's composite is stored to a shared-memory plane SHIFTED by the column's integer shift q_j of
//     this tile (source pixel n lands at output position n - H - q_j; conflict-free scalar stores), double-buffered:
//     one CTA barrier per quad.
//   * Lerp phase: thread i owns the four ADJACENT output pixels m0 + 4 i .. + 3; because of the shifted store the two
//     samples of output pixel o sit at positions o, o + 1 whatever the shift, so a column costs one aligned LDS.128 and
//     one LDS.32: t = a_j c_m - q_j, acc += x0 + t (x1 - x0).  q_j is constant over the tile for ~99 % of the columns
//     (a per-tile table, built once per segment); the rest take a per-pixel floor relative to the stored shift.  Only
//     the shift delta = a_j (lambda0/k + m) is formed in fp32, never the absolute source coordinate.
//   * fp32 column sums are folded into fp64 registers every kFoldPairs pairs; fp64 totals are rounded once on store.
//   * Work = the flattened (star, tile, column pair) list with a cost per pair (bins present + the lerp), cut into
//     equal contiguous ranges, one per CTA (one wave, any number of tiles / stars per CTA, or many CTAs per tile
//     when the spectrum is short).  A tile wholly inside one CTA's range is stored directly (STG.128); a shared
//     tile's fp64 partial sums are added in CTA order by the last CTA to deliver (atomic ticket, self-resetting):
//     run-to-run identical.
//   * Batch (config 5): the same launch walks an array of stars (soap_batch_integrate_quiet).
//   * What bounds it (measured by switching phases off, C3: compute 70 us + lerp 37 us + loads / barriers / store 27 us
//     = 133 us, additive): the shared-memory pipe.  Every thread must receive every weight (4 554 words per tile and
//     thread, 164 KB per quad and SM = 1 280 cycles at 128 B/clk) beside the FFMA2 (1 536 cycles per quad): with 4
//     pixels per thread - what the register file allows - the form is co-bound by LDS bandwidth and the FP32 pipe.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "ptx_helpers.cuh"

namespace soap {
namespace comp {

constexpr int kThreads = 512;
constexpr int kCtasPerSm = 512 / kThreads;  // the register-resident spans fill the register file (2 x 256 and 4 x 128
                                            // threads were measured: within 3 %)
constexpr int kPx = 4;                 // source pixels per thread and mu-bin
constexpr int kSpan = kThreads * kPx;  // source pixels per CTA span
constexpr int kFoldPairs = 4;          // fp32 -> fp64 fold interval (column pairs = 8 columns)
constexpr int kMaxBins = 24;           // mu bins the register-resident form can hold
constexpr int kMaxStars = 256;         // stars per launch
constexpr int kPairCostBase = 24;      // cost model: 8 FFMA2-slots per weight load + the lerp, barrier and loop

struct PairHdr {  // one column pair (2p, 2p+1); entry [n_pairs] carries the total cost in cost0
    float a0, a1;  // shift factors D - 1 of the two columns (0 for the missing column of an odd grid)
    int nl;        // weight loads: bins 0 .. 2 nl - 1 hold every non-zero weight of the pair
    int cost0;     // cost of the pairs before this one
};

struct Star {
    const float *base;   // [n_mu][pitch]
    float *out;          // [n_pix]
    const float2 *Wp;    // [n_pairs][wp_stride]: (W[2p][b], W[2p+1][b])
    const PairHdr *hdr;  // [n_pairs + 1]
    int *ticket;         // [n_tiles] shares delivered per tile; zero between launches
    long long pitch, n_pix, out_lo, out_hi;
    double c0;           // lambda0 / dlambda
    int n_mu, n_pairs, halo, L, n_tiles, wp_stride;
};

struct Params {
    Star one;            // the star of a single-star launch (travels as a kernel argument: no copy)
    const Star *many;    // batch: DEVICE [n_stars]; nullptr = `one`
    int n_stars;
    double *partial;     // [gridDim.x][2][kSpan]
    int max_pairs;       // shared-memory table capacity
    int plane;           // plane_floats(largest halo of the launch)
};

__host__ __device__ inline int plane_floats(int max_halo) { return kSpan + 2 * max_halo + 8; }  // multiple of 4
__host__ __device__ inline size_t smem_bytes(int nb, int max_pairs, int max_halo) {
    return (size_t)2 * 4 * plane_floats(max_halo) * sizeof(float) + (size_t)(max_pairs + 1) * nb * sizeof(float2) +
           (size_t)(max_pairs + 2) * sizeof(PairHdr) + (size_t)(max_pairs + 2) * sizeof(int4) +
           (size_t)(kMaxStars + 1) * sizeof(long long) + sizeof(Star) + 64;
}

// Built by the last CTA of geometry_kernel: the pair tables of the composite form.
__device__ inline void build_composite_tables(int N, int n_mu, const double *col_a, const double *Wbin, float2 *Wp, int wp_stride,
                                              PairHdr *hdr) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
    const int n_pairs = (N + 1) / 2;
    for (int p = warp; p < n_pairs; p += n_warps) {
        const int j0 = 2 * p, j1 = 2 * p + 1;
        int hi = -1;
        for (int b0 = 0; b0 < wp_stride; b0 += 32) {
            const int b = b0 + lane;
            double w0 = 0.0, w1 = 0.0;
            if (b < n_mu) {
                w0 = Wbin[(size_t)j0 * n_mu + b];
                if (j1 < N) w1 = Wbin[(size_t)j1 * n_mu + b];
            }
            if (b < wp_stride) Wp[(size_t)p * wp_stride + b] = make_float2((float)w0, (float)w1);
            const unsigned m = __ballot_sync(0xffffffffu, w0 != 0.0 || w1 != 0.0);
            if (m) hi = b0 + 31 - __clz(m);
        }
        if (lane == 0) {
            PairHdr h;
            h.a0 = (float)col_a[j0];
            h.a1 = j1 < N ? (float)col_a[j1] : 0.f;
            h.nl = (hi + 2) / 2;
            h.cost0 = 0;
            hdr[p] = h;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int p = 0; p < n_pairs; ++p) {
            const int c = 8 * hdr[p].nl + kPairCostBase;
            hdr[p].cost0 = run;
            run += c;
        }
        PairHdr t;
        t.a0 = t.a1 = 0.f;
        t.nl = 0;
        t.cost0 = run;
        hdr[n_pairs] = t;
    }
}

// CTA that owns work unit u when U units are cut into G ranges [floor(g U / G), floor((g+1) U / G)).
__device__ __forceinline__ long long owner_of(long long u, long long U, long long G) { return ((u + 1) * G - 1) / U; }

// Compute phase of one column quad (pairs kk, kk + 1), straight-line for NL weight loads per pair (2 mu bins each) so
// that ptxas hoists the LDS.128 of the next bins above the FFMA2 of the current ones:
// TU[0][r] = (T_j, T_j+1)[pixel r], TU[1][r] = (T_j+2, T_j+3)[pixel r].
template <int NB, int NL>
__device__ __forceinline__ void composite_columns(const float (&S)[NB][kPx], const float4 *__restrict__ w0,
                                                  const float4 *__restrict__ w1, float2 (&TU)[2][kPx]) {
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        const float4 wa = w0[l], wb = w1[l];
#pragma unroll
        for (int r = 0; r < kPx; ++r) TU[0][r] = fma2(make_float2(wa.x, wa.y), bcast2(S[2 * l][r]), TU[0][r]);
#pragma unroll
        for (int r = 0; r < kPx; ++r) TU[1][r] = fma2(make_float2(wb.x, wb.y), bcast2(S[2 * l][r]), TU[1][r]);
#pragma unroll
        for (int r = 0; r < kPx; ++r) TU[0][r] = fma2(make_float2(wa.z, wa.w), bcast2(S[2 * l + 1][r]), TU[0][r]);
#pragma unroll
        for (int r = 0; r < kPx; ++r) TU[1][r] = fma2(make_float2(wb.z, wb.w), bcast2(S[2 * l + 1][r]), TU[1][r]);
    }
}

template <int NB>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) composite_quiet_kernel(const Params p) {
    static_assert(NB % 4 == 0 && NB <= kMaxBins, "bins are loaded two per LDS.128 and unrolled four at a time");
    extern __shared__ __align__(16) unsigned char smem[];
    float *Tbuf = reinterpret_cast<float *>(smem);                                    // [2 buffers][4 columns][plane]
    float2 *Wsm = reinterpret_cast<float2 *>(Tbuf + 2 * 4 * p.plane);                 // [max_pairs + 1][NB]
    PairHdr *hsm = reinterpret_cast<PairHdr *>(Wsm + (size_t)(p.max_pairs + 1) * NB);  // [max_pairs + 2]
    int4 *qtab = reinterpret_cast<int4 *>(hsm + p.max_pairs + 2);                     // [max_pairs + 2] shifts of the current tile
    long long *unit0 = reinterpret_cast<long long *>(qtab + p.max_pairs + 2);         // [n_stars + 1]
    Star *cur = reinterpret_cast<Star *>(unit0 + kMaxStars + 1);
    int *ctl = reinterpret_cast<int *>(cur + 1);                                      // last-CTA flag

    const int tid = threadIdx.x;
    const long long G = gridDim.x, g = blockIdx.x;
    const int n_stars = p.n_stars;

    // (launched with programmatic stream serialization: the pair tables are the geometry launch's, which may still be
    // finishing)
    trigger_dependents();
    grid_dependency_wait();
    // ---- work units of every star: n_tiles x (cost of all its pairs) -------------------------------------------
    for (int s = tid; s < n_stars; s += kThreads) {
        const Star &st = p.many ? p.many[s] : p.one;
        unit0[s + 1] = (long long)st.n_tiles * (long long)__ldcg(&st.hdr[st.n_pairs].cost0);
    }
    __syncthreads();
    if (tid == 0) {
        long long run = 0;
        for (int s = 0; s < n_stars; ++s) {
            const long long c = unit0[s + 1];
            unit0[s] = run;
            run += c;
        }
        unit0[n_stars] = run;
    }
    __syncthreads();
    const long long U = unit0[n_stars];
    if (U <= 0) return;
    const long long B0 = (g * U) / G, B1 = ((g + 1) * U) / G;
    if (B1 <= B0) return;

    int s = 0;
    while (unit0[s + 1] <= B0) ++s;  // the star that holds unit B0 (stars without work are skipped)
    int cur_s = -1;
    long long t = -1;
    int k = 0;
    bool first_seg = true;
    unsigned it = 0;  // column quads processed by this CTA: selects the T buffer

    for (;;) {
        if (s >= n_stars) break;
        if (s != cur_s) {  // ---- this star's tables -> shared memory
            __syncthreads();
            const Star &st = p.many ? p.many[s] : p.one;
            if (tid == 0) *cur = st;
            const int np = st.n_pairs;
            const float4 *src = reinterpret_cast<const float4 *>(st.Wp);
            float4 *dst = reinterpret_cast<float4 *>(Wsm);
            for (int i = tid; i < np * NB / 2; i += kThreads) dst[i] = __ldcg(&src[i]);
            for (int i = tid; i < NB / 2; i += kThreads) dst[np * NB / 2 + i] = make_float4(0.f, 0.f, 0.f, 0.f);  // the pad row
            const int4 *hs = reinterpret_cast<const int4 *>(st.hdr);
            int4 *hd = reinterpret_cast<int4 *>(hsm);
            for (int i = tid; i <= np; i += kThreads) hd[i] = __ldcg(&hs[i]);
            if (tid == 0) hd[np + 1] = make_int4(0, 0, 0, 0);
            cur_s = s;
            __syncthreads();
        }
        const int n_pairs = cur->n_pairs;
        const long long C = hsm[n_pairs].cost0;
        if (first_seg) {  // first pair whose start unit is >= B0
            const long long rel = B0 - unit0[s];
            t = rel / C;
            const int r = (int)(rel - t * C);
            int lo = 0, hi = n_pairs;  // first k with cost0[k] >= r
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (hsm[mid].cost0 >= r) hi = mid;
                else lo = mid + 1;
            }
            k = lo;
            if (k == n_pairs) {
                k = 0;
                ++t;
            }
            first_seg = false;
            if (t >= cur->n_tiles) {
                ++s;
                t = 0;
                continue;
            }
        }
        const long long u_tile = unit0[s] + t * C;
        if (u_tile + hsm[k].cost0 >= B1) break;
        int k_end = n_pairs;
        if (B1 - u_tile < C) {  // first pair whose start unit is >= B1
            const int lim = (int)(B1 - u_tile);
            int lo = k, hi = n_pairs;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (hsm[mid].cost0 >= lim) hi = mid;
                else lo = mid + 1;
            }
            k_end = lo;
        }

        // ================= one segment: pairs [k, k_end) of tile t of star s =======================================
        {
            const int H = cur->halo, L = cur->L, n_mu = cur->n_mu;
            const long long n_pix = cur->n_pix, pitch = cur->pitch;
            const long long m0 = t * (long long)L, n0 = m0 - H;
            const int plane = p.plane;  // floats per column plane of a T buffer: kSpan + 2 H_max + 8
            // ---- the span of every mu-bin row -> registers: thread i holds source pixels n0 + i + kThreads r
            // (clamp-to-edge outside the grid, reading S8)
            float S[NB][kPx];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
#pragma unroll
                for (int r = 0; r < kPx; ++r) {
                    long long nn = n0 + tid + kThreads * r;
                    nn = nn < 0 ? 0 : (nn > n_pix - 1 ? n_pix - 1 : nn);
                    S[b][r] = b < n_mu ? __ldg(cur->base + (long long)b * pitch + nn) : 0.f;
                }
            }
            const float c_first = (float)(cur->c0 + (double)m0), c_last = (float)(cur->c0 + (double)(m0 + L - 1));
            // Integer shifts of this tile, once per (tile, column pair): {qs0, qs1, steady flags, 0}.  Column j's composite is
            // STORED shifted by qs_j (source pixel n lands at output position n - H - qs_j), so the lerp phase reads the two
            // samples of output pixel o at positions o, o + 1 whatever the shift: aligned 16-byte loads of adjacent pixels.
            // qs_j = floor(a_j c) at the tile's first pixel; "steady" = the same at its last pixel (else a per-pixel path
            // corrects by floor(a_j c_o) - qs_j).  Read after the loop's first barrier.
            for (int pp = k + tid; pp < k_end; pp += kThreads) {
                const float a0 = hsm[pp].a0, a1 = hsm[pp].a1;
                const float qf0 = floorf(a0 * c_first), qf1 = floorf(a1 * c_first);
                const int steady = (qf0 == floorf(a0 * c_last) ? 1 : 0) | (qf1 == floorf(a1 * c_last) ? 2 : 0);
                int q0 = (int)qf0, q1 = (int)qf1;
                q0 = max(-(H - 1), min(H - 2, q0));
                q1 = max(-(H - 1), min(H - 2, q1));
                qtab[pp] = make_int4(q0, q1, steady, 0);
            }
            if (tid == 0) qtab[k_end] = make_int4(0, 0, 3, 0);  // the pair after the last (computed, never interpolated)
            // output pixels of this thread: o = 4 tid .. 4 tid + 3 (adjacent: one LDS.128 pair per column, one STG.128)
            const bool valid = 4 * tid < L;
            float c_px[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) c_px[e] = (float)(cur->c0 + (double)(m0 + 4 * tid + e));
            float A[4] = {0.f, 0.f, 0.f, 0.f};
            double tot[4] = {0.0, 0.0, 0.0, 0.0};
            auto compute_quad = [&](int kk, float *buf) {
                // (T_j .. T_j+3)[r] = sum_b W[j..j+3, b] S_b[r]
                const int nl0 = hsm[kk].nl, nl1 = kk + 1 < k_end ? hsm[kk + 1].nl : 0;
                const int nl = max(nl0, nl1);
                float2 TU[2][kPx];
#pragma unroll
                for (int r = 0; r < kPx; ++r) TU[0][r] = TU[1][r] = make_float2(0.f, 0.f);
                const float4 *w0 = reinterpret_cast<const float4 *>(Wsm + (size_t)kk * NB);
                const float4 *w1 = reinterpret_cast<const float4 *>(Wsm + (size_t)(kk + 1) * NB);
                const int step = (nl + 1) >> 1;  // variants of 2, 4, ... weight loads per pair
                if (NB >= 4 && step <= 1) composite_columns<NB, (2 < NB / 2 ? 2 : NB / 2)>(S, w0, w1, TU);
                else if (NB >= 8 && step == 2) composite_columns<NB, (4 < NB / 2 ? 4 : NB / 2)>(S, w0, w1, TU);
                else if (NB >= 12 && step == 3) composite_columns<NB, (6 < NB / 2 ? 6 : NB / 2)>(S, w0, w1, TU);
                else if (NB >= 16 && step == 4) composite_columns<NB, (8 < NB / 2 ? 8 : NB / 2)>(S, w0, w1, TU);
                else if (NB >= 20 && step == 5) composite_columns<NB, (10 < NB / 2 ? 10 : NB / 2)>(S, w0, w1, TU);
                else composite_columns<NB, NB / 2>(S, w0, w1, TU);
                // source pixel (local index tid + kThreads r) of column j -> position tid + kThreads r + H - qs_j  (>= 1)
                const int4 qa = qtab[kk], qb = qtab[kk + 1];
                float *d0 = buf + 0 * plane + tid + H - qa.x, *d1 = buf + 1 * plane + tid + H - qa.y;
                float *d2 = buf + 2 * plane + tid + H - qb.x, *d3 = buf + 3 * plane + tid + H - qb.y;
#pragma unroll
                for (int r = 0; r < kPx; ++r) {
                    d0[kThreads * r] = TU[0][r].x;
                    d1[kThreads * r] = TU[0][r].y;
                    d2[kThreads * r] = TU[1][r].x;
                    d3[kThreads * r] = TU[1][r].y;
                }
            };
            auto lerp_quad = [&](int kk, const float *buf) {
                // A[e] += lerp(T_j; m + a_j c_m) for the (up to) four columns; output pixel o reads positions o + 2 H (+ 1)
                if (!valid) return;
#pragma unroll
                for (int cidx = 0; cidx < 4; ++cidx) {
                    const int pr = cidx >> 1;
                    if (pr == 1 && kk + 1 >= k_end) break;  // the second pair belongs to the next CTA
                    const float a = (cidx & 1) ? hsm[kk + pr].a1 : hsm[kk + pr].a0;
                    const int4 qq = qtab[kk + pr];
                    const int qs = (cidx & 1) ? qq.y : qq.x;
                    const float *pl = buf + cidx * plane + 2 * H + 4 * tid;
                    if (qq.z & (1 << (cidx & 1))) {
                        const float4 v0 = *reinterpret_cast<const float4 *>(pl);
                        const float x4 = pl[4];
                        const float nq = -(float)qs;
                        const float x[5] = {v0.x, v0.y, v0.z, v0.w, x4};
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const float tt = fmaf(a, c_px[e], nq);
                            A[e] += fmaf(tt, x[e + 1] - x[e], x[e]);
                        }
                    } else {  // the integer shift changes inside the tile: per-pixel floor, relative to the stored shift
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const float qf = floorf(a * c_px[e]);
                            const float tt = fmaf(a, c_px[e], -qf);
                            int q = (int)qf;
                            q = max(-(H - 1), min(H - 2, q));
                            const float x0 = pl[e + q - qs], x1 = pl[e + q - qs + 1];
                            A[e] += fmaf(tt, x1 - x0, x0);
                        }
                    }
                }
            };
            int since_fold = 0;
            __syncthreads();  // the shift table is complete
            compute_quad(k, Tbuf + (it & 1u) * (4 * plane));
            for (int kk = k; kk < k_end; kk += 2, ++it) {
                __syncthreads();  // quad kk is in its buffer; the other buffer is free
                float *buf = Tbuf + (it & 1u) * (4 * plane), *nxt = Tbuf + ((it + 1u) & 1u) * (4 * plane);
                if (kk + 2 < k_end) compute_quad(kk + 2, nxt);
                lerp_quad(kk, buf);
                if (++since_fold == kFoldPairs / 2) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        tot[e] += (double)A[e];
                        A[e] = 0.f;
                    }
                    since_fold = 0;
                }
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) tot[e] += (double)A[e];

            // ---- a6: store.  A tile wholly inside this CTA's range goes straight out; otherwise the shares are added
            // in CTA order by the last CTA to deliver.
            const bool whole = k == 0 && k_end == n_pairs;
            const long long lo = cur->out_lo, hi = cur->out_hi < n_pix ? cur->out_hi : n_pix;
            float *out = cur->out;
            const bool vec_ok = (reinterpret_cast<uintptr_t>(out) & 15) == 0;
            const long long m = m0 + 4 * tid;
            if (whole) {
                if (valid) {
                    if (vec_ok && m >= lo && m + 3 < hi) {
                        *reinterpret_cast<float4 *>(out + m) = make_float4((float)tot[0], (float)tot[1], (float)tot[2], (float)tot[3]);
                    } else {
#pragma unroll
                        for (int q = 0; q < 4; ++q)
                            if (m + q >= lo && m + q < hi) out[m + q] = (float)tot[q];
                    }
                }
                __syncthreads();  // every lerp of this segment has read its T buffer and the shift table
            } else {
                const long long u_last = u_tile + hsm[n_pairs - 1].cost0;
                const long long g_first = owner_of(u_tile, U, G), g_last = owner_of(u_last, U, G);
                const int slot = g == g_first ? 1 : 0;  // a CTA's head share (k == 0) and tail share (k > 0) of two tiles
                double *mine = p.partial + ((size_t)g * 2 + slot) * kSpan + 4 * tid;
                reinterpret_cast<double2 *>(mine)[0] = make_double2(tot[0], tot[1]);
                reinterpret_cast<double2 *>(mine)[1] = make_double2(tot[2], tot[3]);
                __threadfence();
                __syncthreads();
                if (tid == 0) {
                    const int ticket = atomicAdd(&cur->ticket[t], 1);
                    const bool last = ticket == (int)(g_last - g_first);
                    if (last) cur->ticket[t] = 0;  // ready for the next launch
                    ctl[0] = last ? 1 : 0;
                }
                __syncthreads();
                if (ctl[0]) {
                    __threadfence();
                    if (valid) {
                        double sum[4] = {0.0, 0.0, 0.0, 0.0};
                        const double *src0 = p.partial + 4 * tid;
                        long long c = g_first;
                        for (; c + 3 <= g_last; c += 4) {  // four shares in flight; added in CTA order
                            double2 v[4][2];
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                const double *src = src0 + ((size_t)(c + u) * 2 + ((c + u) == g_first ? 1 : 0)) * kSpan;
                                v[u][0] = __ldcg(reinterpret_cast<const double2 *>(src));
                                v[u][1] = __ldcg(reinterpret_cast<const double2 *>(src) + 1);
                            }
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                sum[0] += v[u][0].x;
                                sum[1] += v[u][0].y;
                                sum[2] += v[u][1].x;
                                sum[3] += v[u][1].y;
                            }
                        }
                        for (; c <= g_last; ++c) {
                            const double *src = src0 + ((size_t)c * 2 + (c == g_first ? 1 : 0)) * kSpan;
                            const double2 v0 = __ldcg(reinterpret_cast<const double2 *>(src));
                            const double2 v1 = __ldcg(reinterpret_cast<const double2 *>(src) + 1);
                            sum[0] += v0.x;
                            sum[1] += v0.y;
                            sum[2] += v1.x;
                            sum[3] += v1.y;
                        }
                        if (vec_ok && m >= lo && m + 3 < hi) {
                            *reinterpret_cast<float4 *>(out + m) = make_float4((float)sum[0], (float)sum[1], (float)sum[2], (float)sum[3]);
                        } else {
#pragma unroll
                            for (int q = 0; q < 4; ++q)
                                if (m + q >= lo && m + q < hi) out[m + q] = (float)sum[q];
                        }
                    }
                }
                __syncthreads();  // ctl may be rewritten by the next segment
            }
        }

        if (k_end < n_pairs) break;  // the range ends inside this tile
        k = 0;
        if (++t >= cur->n_tiles) {
            ++s;
            t = 0;
        }
    }
}

}  // namespace comp
}  // namespace soap
