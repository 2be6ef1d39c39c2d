// Resolution lowering (Alg. 2, Alg. 5; reading R-LSF):
// every spectrum row is convolved with a Gaussian line-spread function of FWHM lambda / R sampled on the pixel
// grid, per output pixel m:
//   sigma_m = lambda_m / (R 2 sqrt(2 ln 2)),  g_m(j) = exp(-(j k)^2 / (2 sigma_m^2)),  |j| <= J_m = ceil(nsig sigma_m / k),
//   out[m] = sum_j g_m(j) in[clamp(m + j)] / sum_j g_m(j).
//
// The kernel is HBM-bound (one read and one write of every row; ~20 FMAs per pixel).  A thread owns one pixel
// of a 256-pixel tile for ALL rows: its normalised weights (fp64 exp, rounded once to the I/O type) are computed
// once (two exponentials and a product recurrence) and kept in shared memory ([tap][thread]: conflict-free),
// then row after row the tile plus its halo is staged in shared memory with coalesced loads (double-buffered: the
// next row is in flight while this one is computed) and every thread adds its symmetric taps from the outside in.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "ptx_helpers.cuh"

namespace soap {

constexpr int kLsfThreads = 256;
constexpr int kLsfMaxJ = 96;      // taps on each side the kernel supports (host checks)
constexpr int kLsfBreaks = 16;
constexpr double kLsfNsig = 5.0;  // truncation in sigmas (reading R-LSF); the oracle uses the same constant

struct LsfArgs {
    const void *in;
    void *out;
    long long n_rows, n_pix, in_pitch, out_pitch;
    double lambda0, k, R, fwhm_to_sigma;
    int J_max;  // J of the last pixel (sigma grows with lambda): halo of every tile
    // lower_resolution_p_kernel: the half-width J(m) = ceil(5 sigma_m / k) is a non-decreasing step function of the pixel;
    // the host evaluates the defining expression (the same IEEE operations) at the steps only:
    // J(m) = jm0 + #{b : jm_break[b] <= m}; at most kLsfBreaks steps, as the kernel serves J <= 16.
    int jm0, n_breaks;
    long long jm_break[kLsfBreaks];
    double h_scale;  // (k R / fwhm_to_sigma)^2 / 2: k^2 / (2 sigma_m^2) = h_scale / lambda_m^2
};

__host__ __device__ inline size_t lsf_smem_bytes(int J_max, size_t elem) {
    return ((size_t)(J_max + 1) * kLsfThreads + 2 * (size_t)(kLsfThreads + 2 * J_max)) * elem;  // weights + 2 row tiles
}

template <typename T>
__global__ void __launch_bounds__(kLsfThreads) lower_resolution_kernel(const LsfArgs a) {
    extern __shared__ __align__(16) unsigned char lsf_smem[];
    T *w = reinterpret_cast<T *>(lsf_smem);            // [J_max + 1][kLsfThreads]
    T *s = w + (size_t)(a.J_max + 1) * kLsfThreads;    // [kLsfThreads + 2 J_max]
    const int tid = threadIdx.x, J = a.J_max;
    const long long m0 = (long long)blockIdx.x * kLsfThreads;
    const long long m = m0 + tid;
    // ---- this pixel's weights -------------------------------------------------------------------------
    int Jm = 0;
    if (m < a.n_pix) {
        const double lam = __dadd_rn(a.lambda0, __dmul_rn(a.k, (double)m));
        const double sigma = __dmul_rn(__ddiv_rn(lam, a.R), a.fwhm_to_sigma);
        Jm = (int)ceil(__ddiv_rn(__dmul_rn(kLsfNsig, sigma), a.k));
        Jm = min(Jm, J);
        // g(j) = exp(-j^2 h), h = k^2 / (2 sigma^2): g(j+1) = g(j) rho_j with rho_j = rho_{j-1} exp(-2h), rho_0 = exp(-h)
        // (two exponentials per pixel instead of J; the products round to ~J ulp of fp64)
        const double h = (a.k * a.k) / (2.0 * sigma * sigma);
        const double q = exp(-2.0 * h);
        double rho = exp(-h), g = 1.0, norm = 1.0;
        for (int j = 1; j <= Jm; ++j) {
            g *= rho;
            rho *= q;
            norm += 2.0 * g;
        }
        const double inv = 1.0 / norm;
        rho = exp(-h);
        g = 1.0;
        for (int j = 0; j <= J; ++j) {
            w[(size_t)j * kLsfThreads + tid] = j <= Jm ? (T)(g * inv) : (T)0;
            g *= rho;
            rho *= q;
        }
    }
    // ---- rows --------------------------------------------------------------------------------------------
    const T *in = static_cast<const T *>(a.in);
    T *out = static_cast<T *>(a.out);
    // double-buffered row tiles: the next row's samples are in flight (registers) while this row is computed
    const int span = kLsfThreads + 2 * J;
    constexpr int kPer = (kLsfThreads + 2 * kLsfMaxJ + kLsfThreads - 1) / kLsfThreads;  // samples a thread stages
    auto fetch = [&](long long r, T (&v)[kPer]) {
        const T *row = in + r * a.in_pitch;
#pragma unroll
        for (int u = 0; u < kPer; ++u) {
            const int qq = tid + u * kLsfThreads;
            long long n = m0 - J + qq;
            n = n < 0 ? 0 : (n > a.n_pix - 1 ? a.n_pix - 1 : n);  // ends clamped (reading S8)
            v[u] = qq < span ? row[n] : (T)0;
        }
    };
    auto stage = [&](T *dst, const T (&v)[kPer]) {
#pragma unroll
        for (int u = 0; u < kPer; ++u) {
            const int qq = tid + u * kLsfThreads;
            if (qq < span) dst[qq] = v[u];
        }
    };
    T v[kPer];
    long long r = blockIdx.y;
    if (r < a.n_rows) {
        fetch(r, v);
        stage(s, v);
    }
    int cur = 0;
    __syncthreads();  // weights and the first tile are in place
    for (; r < a.n_rows; r += gridDim.y) {
        const long long rn = r + gridDim.y;
        if (rn < a.n_rows) fetch(rn, v);
        if (m < a.n_pix) {
            const T *c = s + (size_t)cur * span + J + tid;
            T acc0 = (T)0, acc1 = (T)0;  // two chains, both from the small outer taps inward
            int j = Jm;
            if (j & 1) {
                acc1 = w[(size_t)j * kLsfThreads + tid] * (c[-j] + c[j]);
                --j;
            }
#pragma unroll 2
            for (; j >= 2; j -= 2) {
                acc0 += w[(size_t)j * kLsfThreads + tid] * (c[-j] + c[j]);
                acc1 += w[(size_t)(j - 1) * kLsfThreads + tid] * (c[-(j - 1)] + c[j - 1]);
            }
            out[r * a.out_pitch + m] = (acc0 + acc1) + w[tid] * c[0];
        }
        if (rn < a.n_rows) stage(s + (size_t)(cur ^ 1) * span, v);
        cur ^= 1;
        __syncthreads();
    }
}

// ---- fp32 fast path -------------------------------------------------------------------------------------------
// The generic kernel above issues ~200 instructions per output pixel (one shared-memory load per sample and per
// weight).  Here a thread owns 4 consecutive pixels of a 1024-pixel tile: its sample window (4 + 2 J4 floats, J4 =
// taps per side rounded up to a multiple of 4, a template parameter so that the window lives in registers) is read
// with LDS.128, the 4 x (J4 + 1) weights stay in registers (from shared memory they would cost two thirds of the
// shared-memory bandwidth and bind the kernel), and rows are written with 16-byte stores: ~30 instructions per output.  Persistent CTAs walk a contiguous range of (tile, row) items in tile-major order,
// so the per-pixel weights (exact, as above) are recomputed only when the tile changes, and the next item's tile
// is in flight while the current one is computed.  Requires 16-byte aligned rows (pitch % 4 == 0).
constexpr int kLsfV = 4;
constexpr int kLsfTileV = kLsfThreads * kLsfV;
constexpr int kLsfStages = 8;  // row tiles in flight per CTA (cp.async ring): ~60 KB per SM in flight covers the HBM latency

template <int J4>
__host__ __device__ constexpr size_t lsf_v_smem_bytes() {
    return kLsfStages * (size_t)(kLsfTileV + 2 * J4) * sizeof(float);
}

template <int J4>
__global__ void __launch_bounds__(kLsfThreads, J4 <= 16 ? 2 : 1) lower_resolution_v_kernel(const LsfArgs a) {
    extern __shared__ __align__(16) unsigned char lsf_smem[];
    float *s = reinterpret_cast<float *>(lsf_smem);  // [kLsfStages][kLsfTileV + 2 J4]
    float wr[J4 + 1][kLsfV];                         // this thread's weights: registers (shared memory would bind)
    constexpr int span = kLsfTileV + 2 * J4, span4 = span / 4;
    constexpr int kPer = (span4 + kLsfThreads - 1) / kLsfThreads;
    const int tid = threadIdx.x;
    const float *in = static_cast<const float *>(a.in);
    float *out = static_cast<float *>(a.out);
    const long long n_tiles = (a.n_pix + kLsfTileV - 1) / kLsfTileV;
    const long long items = n_tiles * a.n_rows;
    const long long it0 = items * blockIdx.x / gridDim.x, it1 = items * (blockIdx.x + 1) / gridDim.x;
    if (it0 >= it1) return;

    // asynchronous 16-byte copies straight into the ring (inner tiles); end tiles are clamped by hand (reading S8)
    // (tile, row) cursors advance by increments: no 64-bit divisions in the loops
    struct Cursor {
        long long it;
        int tile, r;
    };
    auto advance = [&](Cursor &c) {
        ++c.it;
        if (++c.r == (int)a.n_rows) {
            c.r = 0;
            ++c.tile;
        }
    };
    auto issue = [&](const Cursor &ci, float *dst) {
        if (ci.it < it1) {
            const long long tile = ci.tile, r = ci.r;
            const long long g0 = tile * kLsfTileV - J4;  // global pixel of tile-array position 0 (multiple of 4)
            const float *row = in + r * a.in_pitch;
            const bool inner = g0 >= 0 && g0 + span <= a.n_pix;
#pragma unroll
            for (int u = 0; u < kPer; ++u) {
                const int q4 = tid + u * kLsfThreads;
                if (q4 >= span4) continue;
                if (inner || (g0 + 4 * q4 >= 0 && g0 + 4 * q4 + 3 < a.n_pix)) {  // the four pixels lie inside the row
                    cp_async_16(dst + 4 * q4, row + g0 + 4 * q4);
                } else {  // an end tile's out-of-range pixels: clamped by hand
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        long long n = g0 + 4 * q4 + c;
                        n = n < 0 ? 0 : (n > a.n_pix - 1 ? a.n_pix - 1 : n);
                        dst[4 * q4 + c] = row[n];
                    }
                }
            }
        }
        cp_async_commit();  // one group per item, empty or not: the wait below counts groups
    };
    auto weights = [&](long long tile) {  // exact per-pixel weights of this thread's 4 pixels (see the generic kernel)
#pragma unroll
        for (int p = 0; p < kLsfV; ++p) {
            const long long m = tile * kLsfTileV + kLsfV * tid + p;
            const double lam = __dadd_rn(a.lambda0, __dmul_rn(a.k, (double)m));
            const double sigma = __dmul_rn(__ddiv_rn(lam, a.R), a.fwhm_to_sigma);
            int Jm = (int)ceil(__ddiv_rn(__dmul_rn(kLsfNsig, sigma), a.k));
            Jm = min(Jm, J4);
            const double h = (a.k * a.k) / (2.0 * sigma * sigma);
            const double rho0 = exp(-h), q = rho0 * rho0;  // exp(-2h) to 1 ulp of fp64
            // one pass: the unnormalised taps go to the registers as they are formed (fp64 recurrence, rounded once),
            // the norm is summed in fp64, and the taps are scaled by the rounded reciprocal afterwards (one more fp32
            // rounding per tap: 6e-8 relative, far inside the fp32 path's tolerance)
            double rho = rho0, g = 1.0, norm = 1.0;
            wr[0][p] = 1.f;
#pragma unroll
            for (int j = 1; j <= J4; ++j) {
                g *= rho;
                rho *= q;
                const bool in = j <= Jm;
                wr[j][p] = in ? (float)g : 0.f;
                norm += in ? 2.0 * g : 0.0;
            }
            const float inv = (float)(1.0 / norm);
#pragma unroll
            for (int j = 0; j <= J4; ++j) wr[j][p] *= inv;
        }
    };

    Cursor cc, ci;  // compute and issue cursors
    cc.it = it0;
    cc.tile = (int)(it0 / a.n_rows);
    cc.r = (int)(it0 - (long long)cc.tile * a.n_rows);
    ci = cc;
#pragma unroll 1
    for (int d = 0; d < kLsfStages - 1; ++d) {
        issue(ci, s + (size_t)d * span);
        advance(ci);
    }
    long long cur_tile = cc.tile;
    weights(cur_tile);
    int cur = 0;
    for (; cc.it < it1; advance(cc)) {
        const long long tile = cc.tile, r = cc.r;
        cp_async_wait_group<kLsfStages - 2>();  // this item's tile has landed (for this thread's copies) ...
        __syncthreads();                        // ... and for everyone's; the previous item has been consumed
        if (tile != cur_tile) {  // uniform: the whole CTA moves to the next tile
            weights(tile);
            cur_tile = tile;
        }
        issue(ci, s + (size_t)((cur + kLsfStages - 1) % kLsfStages) * span);
        advance(ci);
        // ---- this thread's window and its 4 outputs ---------------------------------------------------
        float win[kLsfV + 2 * J4];
        const float4 *c4 = reinterpret_cast<const float4 *>(s + (size_t)cur * span) + tid;  // window starts at float 4 tid
#pragma unroll
        for (int u = 0; u < (kLsfV + 2 * J4) / 4; ++u) {
            const float4 t = c4[u];
            win[4 * u] = t.x;
            win[4 * u + 1] = t.y;
            win[4 * u + 2] = t.z;
            win[4 * u + 3] = t.w;
        }
        float acc[kLsfV] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int j = J4; j >= 1; --j) {  // small outer taps first
#pragma unroll
            for (int p = 0; p < kLsfV; ++p) acc[p] = fmaf(wr[j][p], win[J4 + p - j] + win[J4 + p + j], acc[p]);
        }
#pragma unroll
        for (int p = 0; p < kLsfV; ++p) acc[p] = fmaf(wr[0][p], win[J4 + p], acc[p]);
        const long long m = tile * kLsfTileV + kLsfV * tid;
        float *o = out + r * a.out_pitch + m;
        if (m + 3 < a.n_pix) {
            *reinterpret_cast<float4 *>(o) = make_float4(acc[0], acc[1], acc[2], acc[3]);
        } else {
#pragma unroll
            for (int p = 0; p < kLsfV; ++p)
                if (m + p < a.n_pix) o[p] = acc[p];
        }
        cur = (cur + 1) % kLsfStages;
    }
}


// ---- fp32 fast path, rows in pairs -------------------------------------------------------------------------------
// The weights depend on the pixel only, so two rows can share every multiply: a thread owns 2 consecutive pixels of a
// 512-pixel tile for a PAIR of rows, the pair's samples are interleaved in shared memory ((row a, row b) per pixel), its
// window is read with LDS.128 (2 pixels x 2 rows each) and every tap is one packed add and one packed FMA (FADD2 / FFMA2,
// weight in the scalar-broadcast operand) over the two rows: half the floating-point instructions of the kernel above,
// no special case for the end tiles (every staged sample is one clamped 4-byte cp.async) and no index arithmetic in the
// inner part.  Persistent CTAs walk a contiguous range of (tile, row pair) items in tile-major order as above.
// Used when the LSF is at most 16 taps per side (the window and the weights must fit in registers).
constexpr int kLsfTileP = kLsfThreads * 2;
constexpr int kLsfStagesP = 8;

template <int J4>
__host__ __device__ constexpr size_t lsf_p_smem_bytes() {
    return kLsfStagesP * (size_t)(kLsfTileP + 2 * J4) * 2 * sizeof(float);
}

template <int J4>
__global__ void __launch_bounds__(kLsfThreads, 3) lower_resolution_p_kernel(const LsfArgs a) {
    static_assert(J4 % 2 == 0, "the window starts on an even pixel");
    extern __shared__ __align__(16) unsigned char lsf_smem[];
    float2 *s = reinterpret_cast<float2 *>(lsf_smem);  // [kLsfStagesP][span] of (row a, row b)
    constexpr int span = kLsfTileP + 2 * J4;
    constexpr int kPer = (span + kLsfThreads - 1) / kLsfThreads;
    float wr[J4 + 1][2];  // this thread's weights: registers
    const int tid = threadIdx.x;
    const float *in = static_cast<const float *>(a.in);
    float *out = static_cast<float *>(a.out);
    const int n_pairs = (int)((a.n_rows + 1) / 2);
    const long long n_tiles = (a.n_pix + kLsfTileP - 1) / kLsfTileP;
    const long long items = n_tiles * n_pairs;
    const long long it0 = items * blockIdx.x / gridDim.x, it1 = items * (blockIdx.x + 1) / gridDim.x;
    if (it0 >= it1) return;

    struct Cursor {
        long long it;
        int tile, rp;
    };
    auto advance = [&](Cursor &c) {
        ++c.it;
        if (++c.rp == n_pairs) {
            c.rp = 0;
            ++c.tile;
        }
    };
    auto issue = [&](const Cursor &ci, float2 *dst) {
        if (ci.it < it1) {
            const long long g0 = (long long)ci.tile * kLsfTileP - J4;  // global pixel of tile-array position 0
            const long long ra = 2LL * ci.rp, rb = ra + 1 < a.n_rows ? ra + 1 : ra;  // an odd last row is paired with itself
            // position q of the tile array holds pixel g0 + q; only the two end tiles need the clamp (reading S8)
            const float *pa = in + ra * a.in_pitch + g0 + tid, *pb = in + rb * a.in_pitch + g0 + tid;
            float2 *d = dst + tid;
            if (g0 >= 0 && g0 + span <= a.n_pix) {
#pragma unroll
                for (int u = 0; u < kPer; ++u) {
                    if (tid + u * kLsfThreads < span) {
                        cp_async_4(&d[u * kLsfThreads].x, pa + u * kLsfThreads);
                        cp_async_4(&d[u * kLsfThreads].y, pb + u * kLsfThreads);
                    }
                }
            } else {
#pragma unroll
                for (int u = 0; u < kPer; ++u) {
                    const int q = tid + u * kLsfThreads;
                    if (q >= span) continue;
                    long long n = g0 + q;
                    n = n < 0 ? 0 : (n > a.n_pix - 1 ? a.n_pix - 1 : n);
                    const int off = (int)(n - g0) - tid;
                    cp_async_4(&d[u * kLsfThreads].x, pa + off);
                    cp_async_4(&d[u * kLsfThreads].y, pb + off);
                }
            }
        }
        cp_async_commit();  // one group per item, empty or not: the wait below counts groups
    };
    // Per-pixel weights of this thread's 2 pixels, once per tile (13 row pairs share them), in fp64: g_j = exp(-h j^2) by the
    // recurrence of the kernels above.  What differs: J(m) comes from the host's step table; h = h_scale / lambda^2 with one
    // reciprocal; the second pixel's exp(-h) is the first's times exp(h - h') by its Taylor series (h - h' ~ 4e-6 h: the
    // cubic term is below 1e-17); 1 / norm by one Newton step from the fp32 reciprocal.  All within a few ulp of fp64:
    // the taps are rounded to fp32 afterwards.
    auto weights = [&](long long tile) {
        const long long m0 = tile * kLsfTileP + 2 * tid;
        int jb = a.jm0, b0 = 0;
        for (; b0 < a.n_breaks && a.jm_break[b0] <= tile * kLsfTileP; ++b0) ++jb;
        const double lam0 = __dadd_rn(a.lambda0, __dmul_rn(a.k, (double)m0));
        const double inv_lam = 1.0 / lam0;
        const double h0 = a.h_scale * inv_lam * inv_lam;
        const double eps = a.k * inv_lam;
        const double dh = h0 * eps * (2.0 - 3.0 * eps);  // h(m0) - h(m0 + 1)
        const double e0 = exp(-h0);
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const long long m = m0 + p;
            int Jm = jb;
            for (int b = b0; b < a.n_breaks && a.jm_break[b] <= m; ++b) ++Jm;
            Jm = min(Jm, J4);
            const double rho0 = p == 0 ? e0 : e0 * (1.0 + dh * (1.0 + 0.5 * dh)), q = rho0 * rho0;
            double rho = rho0, g = 1.0, norm = 1.0;
            wr[0][p] = 1.f;
#pragma unroll
            for (int j = 1; j <= J4; ++j) {
                g *= rho;
                rho *= q;
                const bool inw = j <= Jm;
                wr[j][p] = inw ? (float)g : 0.f;
                norm += inw ? 2.0 * g : 0.0;
            }
            double r = (double)(1.f / (float)norm);
            r = r * (2.0 - norm * r);  // relative error (2^-23)^2
            const float inv = (float)r;
#pragma unroll
            for (int j = 0; j <= J4; ++j) wr[j][p] *= inv;
        }
    };

    Cursor cc, ci;
    cc.it = it0;
    cc.tile = (int)(it0 / n_pairs);
    cc.rp = (int)(it0 - (long long)cc.tile * n_pairs);
    ci = cc;
#pragma unroll 1
    for (int d = 0; d < kLsfStagesP - 1; ++d) {
        issue(ci, s + (size_t)d * span);
        advance(ci);
    }
    long long cur_tile = cc.tile;
    weights(cur_tile);
    int cur = 0;
    for (; cc.it < it1; advance(cc)) {
        const long long tile = cc.tile;
        cp_async_wait_group<kLsfStagesP - 2>();  // this item's samples have landed (for this thread's copies) ...
        __syncthreads();                         // ... and for everyone's; the previous item has been consumed
        if (tile != cur_tile) {
            weights(tile);
            cur_tile = tile;
        }
        issue(ci, s + (size_t)((cur + kLsfStagesP - 1) % kLsfStagesP) * span);
        advance(ci);
        // ---- this thread's window (2 + 2 J4 pixels of both rows) and its 2 x 2 outputs -------------------------------
        float2 win[2 + 2 * J4];
        const float4 *c4 = reinterpret_cast<const float4 *>(s + (size_t)cur * span) + tid;  // window starts at pixel 2 tid
#pragma unroll
        for (int u = 0; u < (2 + 2 * J4) / 2; ++u) {
            const float4 t = c4[u];
            win[2 * u] = make_float2(t.x, t.y);
            win[2 * u + 1] = make_float2(t.z, t.w);
        }
        // two partial sums per pixel (odd and even taps): four independent FFMA2 chains per thread.  From the centre outwards,
        // so that the window's registers are released as the taps are used (77 registers: 3 CTAs per SM).
        float2 acc[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)}, acb[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
        for (int j = 1; j <= J4; ++j) {
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                float2 &t = (j & 1) ? acb[p] : acc[p];
                t = fma2(bcast2(wr[j][p]), add2(win[J4 + p - j], win[J4 + p + j]), t);
            }
        }
#pragma unroll
        for (int p = 0; p < 2; ++p) acc[p] = add2(fma2(bcast2(wr[0][p]), win[J4 + p], acc[p]), acb[p]);
        const long long m = tile * kLsfTileP + 2 * tid;
        const long long ra = 2LL * cc.rp;
        float *oa = out + ra * a.out_pitch + m;
        if (m + 1 < a.n_pix) {
            *reinterpret_cast<float2 *>(oa) = make_float2(acc[0].x, acc[1].x);
            if (ra + 1 < a.n_rows) *reinterpret_cast<float2 *>(oa + a.out_pitch) = make_float2(acc[0].y, acc[1].y);
        } else if (m < a.n_pix) {
            oa[0] = acc[0].x;
            if (ra + 1 < a.n_rows) oa[a.out_pitch] = acc[0].y;
        }
        cur = (cur + 1) % kLsfStagesP;
    }
}

}  // namespace soap
