// a3 + a5 + a6 of SURVEY section 8 for fp32 spectra: the warp-specialised shift-interpolate-accumulate
// kernel (direct form).
//
//   out[m] = sum over entries e of  W_e * lerp(S_row(e); m + delta_e(m)),   delta_e(m) = a_e (lambda0/k + m)
//
// (Alg. 1 / Eq. 3 with Eq. 5-9 written as a gather; see sia.cuh for the
// generic-precision kernel that serves fp64 I/O.)  An entry is a (column, mu-bin) pair with its binned
// weight, or a single cell; entries of a spectrum row are ordered by shift factor a_e.
//
// The path is bound by the FP32 pipe: the 2 FMAs of a lerp-accumulate are the only
// instructions the method needs per (entry, pixel).  Everything here exists to keep every other
// instruction out of the consumers' loop and to keep the four SM sub-partitions equally loaded:
//
//   * CTA = 2 warpgroups: warps 0-3 consume, warps 4-7 produce.  Warp w runs on sub-partition w % 4, so
//     every sub-partition holds one consumer and one producer warp of each resident CTA; `setmaxnreg`
//     moves the producers' registers to the consumers (40 / 120 per thread, 3 CTAs per SM).
//   * A consumer thread owns R = 16 pixels of a 2048-pixel wavelength tile (pixel m_t0 + tid + 128 r:
//     conflict-free shared-memory reads, coalesced stores).
//   * "jobs" = (spectrum row, <= 128 entries) of one tile.  Stage k of the 4-deep ring belongs to producer
//     warp k, which handles jobs k, k+4, ... of the CTA: lane 0 issues two 1-D TMA bulk copies (the span of
//     the row the tile's shifts can reach, and the job's raw entries), then the warp turns the raw entries
//     into what the consumers need:
//       - a record {W, W a} per entry;
//       - a run table: maximal groups of consecutive entries whose integer shift q is the same for every
//         pixel of the tile.  Consumers load their 16 samples and 16 sample differences once per run;
//       - entries whose q changes inside the tile ("flips", ~1 %) become runs of their own and take a
//         per-pixel path.  The producer also writes the clamp-to-edge halo (reading S8) of end tiles;
//       - a descriptor {tile origin, kind, first / last job of the tile, where the result goes}: the
//         consumers are driven by descriptors alone and walk no work list.
//     Full/empty mbarriers per stage; consumers never meet a CTA-wide barrier.
//   * per (entry, thread): 1 LDS.64 (broadcast) + 16 packed FFMA2 (fma.rn.f32x2: two pixels per issue
//     slot) for 16 pixels.  With t = a c - q (c = lambda0/k + m, q the run's integer shift), W lerp =
//     W (s + t d) regroups to W u + (W a) v with u = s - q d and v = c d per pixel of the run: every FMA
//     has one scalar (broadcast) operand, the form that runs at the full lane rate on B200.
//   * precision: only the shift delta (|delta| < ~50) is formed in fp32, never the absolute source
//     coordinate; fp32 partial sums are folded into fp64 every kFold entries.
//   * quiet launch: the flattened (tile, entry) work list is cut into equal contiguous ranges, one per
//     CTA, grid = resident CTA slots (one wave, no tail); a CTA writes one fp64 partial per tile it
//     touches and the last CTA to deliver its share of a tile adds the shares in CTA order (deterministic).
//   * active launch: persistent CTAs take the (star, phase, tile) items, heaviest phase first, from a global
//     counter (active_prepare_kernel builds the per-phase job lists; a CTA's scheduler warp ranks a star's
//     phases by their entry counts); the post-shift contrast (I_ratio of Eq. 3) of a kind multiplies the
//     fp32 partial sums of that kind in fp64 when they are folded into the fp64 totals (a6).
//   * effects launch (EFFECTS): the three outputs of Eq. 1-3 - total, flux only, CB only - from ONE pass over the entries.
//     They are three weightings of the same interpolated sums: with P the fp32 partial sum of a kind (active.cuh lists the
//     kinds) and C the contrast of its region type, every output adds (a + b C) P for a pair (a, b) in {0, 1, -1} that
//     depends on (kind, output) only - Params::eff.  The consumers keep three sets of fp64 totals (208 registers; 2 CTAs per SM).
#pragma once
#include <climits>
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

#include "active.cuh"
#include "ptx_helpers.cuh"

namespace soap {
namespace f32 {

constexpr int kConsumerWarps = 4;
constexpr int kProducerWarps = 4;
constexpr int kConsumers = 32 * kConsumerWarps;             // consumer threads
constexpr int kThreads = kConsumers + 32 * kProducerWarps;  // two warpgroups
constexpr int kR = 16;                                      // pixels per consumer thread
constexpr int kTile = kConsumers * kR;                      // pixels per tile
constexpr int kStages = kProducerWarps;                     // jobs in flight: stage k belongs to producer warp k
constexpr int kJobCap = kActiveJobCap;                      // entries per job (even)
constexpr int kFold = 64;                                   // fp32 -> fp64 fold interval (entries)
constexpr int kFlip = INT_MIN;                              // run marker: per-pixel path
constexpr int kCtasPerSm = 3;
constexpr int kRegsConsumer = 120, kRegsProducer = 40;      // (120 + 40) * 128 = 80 * 256: the launch allocation
constexpr int kCtasPerSmEffects = 2;                        // effects launch: three sets of fp64 totals per consumer thread
constexpr int kRegsConsumerEffects = 208;                   // (208 + 40) * 128 <= 128 * 256
constexpr int kEffKinds = 8;                                // kinds of the effects form (active.cuh)
static_assert(kConsumerWarps == 4 && kProducerWarps == 4, "setmaxnreg acts on aligned groups of 4 warps");

enum : int { kJobFirst = 1, kJobLast = 2, kJobExit = 4 };

// What a launch needs to know about one star.  The quiet launch carries one as a kernel argument; the active launch
// reads a DEVICE array of them, one per star of the batch (soap_batch_active_timeseries: ONE launch for all stars).
struct StarBlock {
    const float *base[3];      // spectrum tables per kind (quiet launch: base[0] only)
    const float *contrast[3];  // per-pixel multiplier per kind or nullptr (== 1); kind 0 unused
    long long pitch, n_pix;
    long long out_lo, out_hi;  // only pixels out_lo <= m < out_hi are stored (0, n_pix; narrower for a window whose margins
                               // belong to its neighbours, see soap_synthesize_host)
    long long row_len;         // elements of a row that may be read from its first pixel on (<= pitch; the pitch itself
                               // unless the table is a window into a wider one, see soap_synthesize_host)
    long long out_pitch;
    double c0;                 // lambda0 / dlambda
    const float2 *ent;         // raw entries (a_e, W_e)
    float *out;                // quiet: [n_pix]; active: [n_phases][out_pitch]; effects launch: the total (nullable)
    float *out_fc[2];          // effects launch: flux-only and CB-only outputs (nullable)
    // active launch
    const ActiveJob *jobs;     // [n_phases][job_cap]
    const int *n_jobs;         // [n_phases]
    const int *work;           // [n_phases] entries of every phase: the launch takes the heaviest phases first
    long long item0;           // first (phase, tile) item of this star in the launch's item list
    int halo;                  // H: multiple of 4, >= max |delta| + 2
    int n_mu, n_tiles, job_cap, n_phases, pad;
};
static_assert(sizeof(StarBlock) % 16 == 0 && sizeof(StarBlock) <= 192, "producer warps cache a block with 16-byte copies");

constexpr int kMaxBatchStars = 96;   // stars per active launch (their item offsets live in shared memory)

struct Params {
    StarBlock one;             // quiet launch, and active launch of a single star: the star (no copy: a kernel argument)
    const StarBlock *many;     // active launch of a batch: DEVICE [n_stars]; nullptr = `one`
    int n_stars;
    long long n_items;         // active launch: (phase, tile) items of all stars
    int halo;                  // largest halo of the launch: sizes the stages
    int stage_bytes, raw_off, rec_off, run_off, desc_off;  // stage_layout(halo), filled by set_layout()
    int collapse;              // SOAP_FORM_FIR: a run's entries are summed into one record {sum W, sum W a}
    // quiet launch
    const int *row_start;      // [n_mu + 1] entry offsets (even)
    double *partial;           // [gridDim.x][max_seg][kTile]
    int max_seg;
    int *tile_ticket;          // [n_tiles] shares delivered per tile; zero between launches
    // active launch
    int *item_counters;        // [2] item hand-out (zero between launches)
    int item_chunk;            // items a CTA takes per hand-out (1 unless the list is very long: a batch of stars)
    int order_phases;          // active launch: take a star's phases heaviest first (0: as given)
    // effects launch, per kind: bits 0-1 spectrum table (0 quiet, 1 spot, 2 facula), bits 2-3 region type whose contrast C
    // applies (0: none), then for output o = 0 total, 1 flux only, 2 CB only two bits at 4 + 2 o: the multiplier of the
    // kind's partial sum - 0: 0, 1: 1, 2: C, 3: 1 - C
    int eff[kEffKinds];
};
enum : int { kMulZero = 0, kMulOne = 1, kMulC = 2, kMulOneMinusC = 3 };
__host__ __device__ constexpr int eff_code(int table, int ctype, int m_total, int m_flux, int m_cb) {
    return table | (ctype << 2) | (m_total << 4) | (m_flux << 6) | (m_cb << 8);
}

// __ldcg of a pointer-valued field
template <typename P>
__device__ __forceinline__ P *ldg_ptr(P *const *addr) {
    return reinterpret_cast<P *>(__ldcg(reinterpret_cast<const unsigned long long *>(addr)));
}

template <bool ACTIVE>
__device__ __forceinline__ const StarBlock &star_block(const Params &p, int star) {
    if (ACTIVE) return p.many[star];
    return p.one;
}

// First unit of CTA c when U units (U even) are cut into G contiguous ranges with even boundaries.
__host__ __device__ inline long long range_begin(long long c, long long U, long long G) {
    return 2 * ((c * (U / 2)) / G);
}

__host__ __device__ constexpr int span_px(int halo) { return kTile + 2 * halo + 4; }

struct Desc {  // written by the producer with the rest of the stage
    long long m_t0;  // first pixel of the tile
    int flags, kind, out_idx, n_runs;
    // active launch: what the consumers need to know about the item's star (a batch mixes stars)
    int star, halo;
    double c0;
    long long out_lo, out_hi, out_pitch;
    float *out;
    float *out_fc[2];          // effects launch
    const float *contrast[2];  // of region types 1, 2
};

struct StageLayout {
    size_t row_bytes, raw_off, rec_off, run_off, desc_off, stage_bytes;
};
__host__ __device__ inline StageLayout stage_layout(int halo) {
    StageLayout l;
    l.row_bytes = ((size_t)span_px(halo) * sizeof(float) + 127) & ~(size_t)127;
    l.raw_off = l.row_bytes;
    l.rec_off = l.raw_off + kJobCap * sizeof(float2);
    l.run_off = l.rec_off + (kJobCap + 2) * sizeof(float2);
    l.desc_off = (l.run_off + (kJobCap + 2) * sizeof(int2) + 15) & ~(size_t)15;
    l.stage_bytes = (l.desc_off + sizeof(Desc) + 127) & ~(size_t)127;
    return l;
}
constexpr size_t kPrefixOff = 1280;                           // active launch: first item of every star, [kMaxBatchStars + 1]
constexpr size_t kBlockCacheOff = 2176;                       // active launch: the star block each producer warp works on
constexpr size_t kBlockCacheStride = 192;                     // >= sizeof(StarBlock), multiple of 16
constexpr int kOrderCap = 256;                                // phases of one star the scheduler orders by work (more: as given)
constexpr size_t kOrderOff = 3072;                            // active launch, scheduler warp: order and jobs of the phases of one
                                                              // star, [kOrderCap] unsigned short each
constexpr size_t kHeaderBytes = 3072 + kOrderCap * 4;         // mbarriers (96 B), tile hand-over words, item queue (at 128), prefix, blocks, order
constexpr size_t kFinBytes = (size_t)kTile * sizeof(float);  // active launch: staged contrast of the current kind
__host__ inline size_t smem_bytes(int halo, bool active) {
    return kHeaderBytes + (active ? kFinBytes : 0) + kStages * stage_layout(halo).stage_bytes;
}

inline void set_layout(Params &p) {  // host: the stage layout travels as kernel arguments (constant bank)
    const StageLayout l = stage_layout(p.halo);
    p.stage_bytes = (int)l.stage_bytes;
    p.raw_off = (int)l.raw_off;
    p.rec_off = (int)l.rec_off;
    p.run_off = (int)l.run_off;
    p.desc_off = (int)l.desc_off;
}

struct Job {
    long long tile;
    int star;
    int kind, row;
    int begin;  // first entry (global index, even)
    int count;  // entries, <= kJobCap (0: an item without entries)
    int flags, out_idx;
};

// ---- job sources: the n-th job of this CTA (every lane of a producer warp computes the same answer) ----------
enum : int { kSrcJob = 0, kSrcExit = 1, kSrcBeyond = 2 };

// Quiet launch: CTA c owns units [range_begin(c), range_begin(c+1)) of the flattened (tile, entry) list; the
// entries of a tile are contiguous (rows back to back), so a job is a chunk of one row inside that range.
struct QuietSource {
    const int *row_start;
    long long E, u0, u1, t, t_first;
    int e, e_lo, e_hi, s, cur;
    bool done;
    __device__ void init(const Params &p, long long cta, long long G) {
        row_start = p.row_start;
        E = __ldcg(&row_start[p.one.n_mu]);
        const long long U = E * p.one.n_tiles;
        u0 = range_begin(cta, U, G);
        u1 = range_begin(cta + 1, U, G);
        done = u1 <= u0;
        t = t_first = done ? 0 : u0 / E;
        cur = 0;
        open_tile();
    }
    __device__ void open_tile() {
        const long long lo = u0 - t * E, hi = u1 - t * E;
        e_lo = (int)(lo > 0 ? lo : 0);
        e_hi = (int)(hi < E ? hi : E);
        e = e_lo;
        s = 0;
    }
    __device__ bool next(Job &j) {
        if (done) return false;
        while (e >= e_hi) {
            ++t;
            if (t * E >= u1) {
                done = true;
                return false;
            }
            open_tile();
        }
        while (__ldcg(&row_start[s + 1]) <= e) ++s;  // rows without entries are skipped
        const int end = min(min(e + kJobCap, __ldcg(&row_start[s + 1])), e_hi);
        j.tile = t;
        j.star = 0;
        j.kind = 0;
        j.row = s;
        j.begin = e;
        j.count = end - e;
        j.flags = (e == e_lo ? kJobFirst : 0) | (end == e_hi ? kJobLast : 0);
        j.out_idx = (int)(t - t_first);
        e = end;
        return true;
    }
    __device__ int get(int n, Job &j) {
        while (cur <= n) {
            if (!next(j)) return n == cur ? kSrcExit : kSrcBeyond;
            ++cur;
        }
        return kSrcJob;
    }
};

// Active launch: items = (phase, tile), ordered heaviest phase first, handed out through one global counter:
// a CTA takes the next item whenever its producers run short of jobs (heaviest-first list scheduling: the
// CTAs finish within one small item of each other).  Which CTA computes an item does not change its result,
// so the output stays run-to-run identical.  Producer warp 0 is the CTA's scheduler: it fetches item numbers
// and publishes (item, first job number) in a small shared-memory ring that the four producer warps read in
// step; it stays kQueueAhead jobs ahead of its own position.  An item's jobs are its phase's job list applied
// to its tile; a phase without covered cells yields one empty job so that its zeros are written (S19).
constexpr int kQueueSlots = 64;  // items in flight per CTA: the producers are never more than ~16 jobs apart, a hand-out <= 16 items
constexpr int kQueueAhead = 2 * kStages;
constexpr int kMaxItemChunk = 16;
struct ItemQueue {               // shared memory
    int4 slot[kQueueSlots];      // {number of the item's first job, phase (-1 = no more items), tile, jobs of the phase << 8 | star}
    int tail;                    // items published
};
static_assert(kMaxBatchStars <= 256, "the star index travels in 8 bits of a queue slot");

struct ActiveSource {
    const StarBlock *many;
    const long long *prefix;  // shared memory: first item of every star, prefix[n_stars] = n_items
    int *counters;  // [0] next item, [1] CTAs that finished fetching (both zero between launches)
    ItemQueue *queue;
    StarBlock *cache;  // shared memory: this warp's copy of the block of the star it is working on
    unsigned short *s_order;    // scheduler: the phases of star `ord_star`, heaviest first (ties by phase index)
    unsigned short *s_njobs;    // scheduler: jobs of its phases
    int ord_star;
    bool ord_identity;          // more than kOrderCap phases: taken as given
    long long n_items;
    int n_stars, chunk;
    bool scheduler, order;
    int pub, pub_end;  // scheduler: items published, job number after the last of them
    bool pub_done;
    int cs_pub;        // scheduler: star of the last hand-out's first item (item numbers only grow)
    int cached_star;
    int i;             // item this warp is working through
    int n0, nj, cnt, phase, tile, star;
    bool done;
    // scheduler warp: the phases of star `st` ordered by work, heaviest first (list scheduling: the CTAs then finish within
    // one small item of each other).  Which CTA computes an item, and when, does not change its result.
    __device__ void load_order(int st) {
        const int lane = threadIdx.x & 31;
        const StarBlock *b = many ? many + st : cache;
        const int n = many ? __ldcg(&b->n_phases) : b->n_phases;
        const int *wk = many ? ldg_ptr(&b->work) : b->work, *njp = many ? ldg_ptr(&b->n_jobs) : b->n_jobs;
        ord_star = st;
        ord_identity = n > kOrderCap || !order;
        if (ord_identity) return;
        __syncwarp();
        bool wide = false;
        for (int k = lane; k < n; k += 32) {
            const int nj = __ldcg(&njp[k]);
            s_njobs[k] = (unsigned short)nj;
            wide = wide || nj > 0xffff;
        }
        if (__any_sync(0xffffffffu, wide)) {  // job counts beyond 16 bits: taken as given, counts read from global memory
            ord_identity = true;
            return;
        }
        // rank of phase ph = phases that go before it.  The list stays L1-resident: ld.global.ca, which - unlike the read-only
        // path - is coherent with what the active-map launch wrote once the dependency wait has returned
        for (int ph = lane; ph < n; ph += 32) {
            const int w = __ldca(&wk[ph]);
            int rk = 0;
#pragma unroll 4
            for (int q = 0; q < n; ++q) {
                const int wq = __ldca(&wk[q]);
                rk += (wq > w || (wq == w && q < ph)) ? 1 : 0;
            }
            s_order[rk] = (unsigned short)ph;
        }
        __syncwarp();
    }
    // scheduler warp: publish items until they cover job number n_need (or the list is exhausted).  A hand-out takes
    // `chunk` consecutive items; lane l looks up item l of it (star, phase, tile, jobs of the phase).
    __device__ void publish_until(int n_need) {
        const int lane = threadIdx.x & 31;
        while (!pub_done && pub_end <= n_need) {
            int first = 0;
            if (lane == 0) first = atomicAdd(&counters[0], chunk);
            first = __shfl_sync(0xffffffffu, first, 0);
            const long long idx = (long long)first + lane;
            const bool valid = lane < chunk && idx < n_items;
            int ph = -1, tl = 0, c = 0, stx = cs_pub;
            if (valid)
                while (idx >= prefix[stx + 1]) ++stx;
            unsigned todo = __ballot_sync(0xffffffffu, valid);
            while (todo) {  // star by star (a hand-out rarely spans more than one)
                const int st = __shfl_sync(0xffffffffu, stx, __ffs(todo) - 1);
                if (st != ord_star) load_order(st);
                const bool mine = valid && stx == st;
                if (mine) {
                    const StarBlock *b = many ? many + st : cache;
                    const int nt = many ? __ldcg(&b->n_tiles) : b->n_tiles;
                    const long long local = idx - prefix[st];
                    const int k = (int)(local / nt);
                    tl = (int)(local - (long long)k * nt);
                    if (ord_identity) {
                        ph = k;
                        c = __ldcg((many ? ldg_ptr(&b->n_jobs) : b->n_jobs) + ph);
                    } else {
                        ph = s_order[k];
                        c = s_njobs[ph];
                    }
                }
                todo &= ~__ballot_sync(0xffffffffu, mine);
            }
            const int jobs = valid ? (c > 0 ? c : 1) : 0;
            int incl = jobs;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            const int n_valid = __popc(__ballot_sync(0xffffffffu, valid));
            const bool ended = n_valid < chunk;  // the list is exhausted: an end marker follows the last item
            if (valid) queue->slot[(pub + lane) % kQueueSlots] = make_int4(pub_end + incl - jobs, ph, tl, (c << 8) | stx);
            if (ended && lane == n_valid) queue->slot[(pub + lane) % kQueueSlots] = make_int4(pub_end + total, -1, 0, 0);
            if (ended) {
                pub_done = true;
                if (lane == 0 && atomicAdd(&counters[1], 1) == (int)gridDim.x - 1) {  // every CTA has stopped fetching
                    counters[0] = 0;
                    counters[1] = 0;
                }
            }
            __syncwarp();
            if (lane == 0) {
                __threadfence_block();
                *reinterpret_cast<volatile int *>(&queue->tail) = pub + n_valid + (ended ? 1 : 0);
            }
            pub += n_valid + (ended ? 1 : 0);
            pub_end += total;
            cs_pub = __shfl_sync(0xffffffffu, stx, 0);
            __syncwarp();
        }
    }
    __device__ void load_item() {
        const volatile int *tail = reinterpret_cast<const volatile int *>(&queue->tail);
        while (*tail <= i) __nanosleep(20);
        __threadfence_block();
        const volatile int *sl = reinterpret_cast<const volatile int *>(&queue->slot[i % kQueueSlots]);
        n0 = sl[0];
        phase = sl[1];
        tile = sl[2];
        const int w = sl[3];
        done = phase < 0;
        if (done) return;
        cnt = w >> 8;
        star = w & 255;
        nj = cnt > 0 ? cnt : 1;
        if (many && star != cached_star) {  // this warp moves on to another star: copy its block
            const int lane = threadIdx.x & 31;
            __syncwarp();
            if (lane < (int)(sizeof(StarBlock) / 16))
                reinterpret_cast<uint4 *>(cache)[lane] = __ldcg(reinterpret_cast<const uint4 *>(many + star) + lane);
            __syncwarp();
            cached_star = star;
        }
    }
    __device__ void init(const Params &p, ItemQueue *q, const long long *pref, StarBlock *my_cache, bool is_scheduler,
                         unsigned char *order_mem) {
        s_order = reinterpret_cast<unsigned short *>(order_mem);
        s_njobs = s_order + kOrderCap;
        ord_star = -1;
        ord_identity = false;
        many = p.many;
        prefix = pref;
        counters = p.item_counters;
        queue = q;
        cache = my_cache;
        n_items = p.n_items;
        n_stars = p.n_stars;
        chunk = p.item_chunk;
        order = p.order_phases != 0;
        scheduler = is_scheduler;
        pub = 0;
        pub_end = 0;
        pub_done = false;
        cs_pub = 0;
        cached_star = -1;
        if (!many) {  // a single star: its block travels as a kernel argument
            if ((threadIdx.x & 31) == 0) *cache = p.one;
            __syncwarp();
            cached_star = 0;
        }
        i = -1;
        n0 = 0;
        nj = 0;
        star = 0;
        done = false;
    }
    __device__ int get(int n, Job &j) {
        if (scheduler) publish_until(n + kQueueAhead);
        while (!done && n >= n0 + nj) {
            ++i;
            load_item();
        }
        if (done) return n == n0 ? kSrcExit : kSrcBeyond;
        const int k = n - n0;
        j.tile = tile;
        j.star = star;
        j.out_idx = phase;
        if (cnt == 0) {
            j.kind = j.row = j.begin = j.count = 0;
            j.flags = kJobFirst | kJobLast;
        } else {
            const int4 a = __ldca(reinterpret_cast<const int4 *>(cache->jobs + (size_t)phase * cache->job_cap + k));
            j.begin = a.x;
            j.count = a.y;
            j.kind = a.z;
            j.row = a.w;
            j.flags = (k == 0 ? kJobFirst : 0) | (k == cnt - 1 ? kJobLast : 0);
        }
        return kSrcJob;
    }
};

// Barrier among the 128 consumer threads only (the producers never take part).
__device__ __forceinline__ void consumer_bar_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kConsumers) : "memory"); }

__device__ __forceinline__ void mbar_wait_backoff(uint64_t *bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) __nanosleep(40);
}

// One producer warp: turns the `count` raw entries (a, W) of a job into records and the run table of a tile
// whose first / last pixel have lambda0/k + m = c_first / c_last.  Returns the number of runs; runs[n_runs] is
// left to the caller.  Without `collapse`: rec[i] = {W, W a} per entry, runs[k] = (first entry, q or kFlip).
// With it: rec[k] = {sum W, sum W a} over run k, runs[k] = (k, q), and a flip entry keeps (its raw index, kFlip).
__device__ __forceinline__ int build_runs(const float2 *raw, int count, float c_first, float c_last, int H, int collapse,
                                          float2 *rec, int2 *runs) {
    const int lane = threadIdx.x & 31;
                int n_runs = 0, carry = kFlip;  // kFlip never equals a q: the first entry opens a run
                for (int i0 = 0; i0 < count; i0 += 32) {
                    const int i = i0 + lane;
                    const bool valid = i < count;
                    int code = kFlip;
                    float2 r2 = make_float2(0.f, 0.f);
                    if (valid) {
                        const float2 en = raw[i];
                        const float qf = floorf(en.x * c_first), ql = floorf(en.x * c_last);
                        int qi = (int)qf;
                        qi = max(-H, min(H + 2, qi));
                        r2 = make_float2(en.y, en.y * en.x);  // {W, W a}
                        if (!collapse) rec[i] = r2;
                        if (qf == ql) code = qi;
                    }
                    int prev = __shfl_up_sync(0xffffffffu, code, 1);
                    if (lane == 0) prev = carry;
                    const bool start = valid && (code == kFlip || code != prev);
                    const unsigned mask = __ballot_sync(0xffffffffu, start);
                    const int ridx = n_runs + __popc(mask & ((2u << lane) - 1u)) - 1;  // run this entry belongs to
                    if (collapse) {
                        // W lerp = W u + (W a) v is linear in {W, W a} for the fixed u, v of a run: the run's entries
                        // collapse into one record {sum W, sum W a} (exact in exact arithmetic; fixed shuffle tree).
                        // A flip entry keeps its raw index: the consumers read it from `raw`.
                        const unsigned heads = mask | 1u;  // lane 0 heads a segment even when it continues a run
                        const int seg0 = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));  // first lane of my segment
                        const unsigned vmask = __ballot_sync(0xffffffffu, valid);
                        const bool tail = valid && (lane == 31 || !((vmask >> (lane + 1)) & 1u) || ((mask >> (lane + 1)) & 1u));
    #pragma unroll
                        for (int d = 1; d < 32; d <<= 1) {
                            const float tx = __shfl_up_sync(0xffffffffu, r2.x, d), ty = __shfl_up_sync(0xffffffffu, r2.y, d);
                            if (lane - d >= seg0) {
                                r2.x += tx;
                                r2.y += ty;
                            }
                        }
                        if (tail && code != kFlip) {
                            const bool fresh = (mask >> seg0) & 1u;  // the segment opened a run in this batch
                            float2 acc2 = fresh ? make_float2(0.f, 0.f) : rec[ridx];
                            rec[ridx] = make_float2(acc2.x + r2.x, acc2.y + r2.y);
                        }
                        if (start) runs[ridx] = make_int2(code == kFlip ? i : ridx, code);
                        __syncwarp();
                    } else if (start) {
                        runs[ridx] = make_int2(i, code);
                    }
                    n_runs += __popc(mask);
                    carry = __shfl_sync(0xffffffffu, code, 31);
                }
    return n_runs;
}

__device__ __forceinline__ void init_source(QuietSource &src, const Params &p, ItemQueue *, const long long *, StarBlock *, bool,
                                            unsigned char *) {
    src.init(p, blockIdx.x, gridDim.x);
}
__device__ __forceinline__ void init_source(ActiveSource &src, const Params &p, ItemQueue *q, const long long *prefix,
                                            StarBlock *cache, bool is_scheduler, unsigned char *order_mem) {
    src.init(p, q, prefix, cache, is_scheduler, order_mem);
}
__device__ __forceinline__ const StarBlock &source_block(const QuietSource &, const Params &p) { return p.one; }
__device__ __forceinline__ const StarBlock &source_block(const ActiveSource &src, const Params &) { return *src.cache; }

template <bool ACTIVE, bool EFFECTS = false>
__global__ void __launch_bounds__(kThreads, EFFECTS ? kCtasPerSmEffects : kCtasPerSm) sia_f32_kernel(const Params p) {
    static_assert(ACTIVE || !EFFECTS, "the effects form is an active launch");
    constexpr int NOUT = EFFECTS ? 3 : 1;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *bar_tma = reinterpret_cast<uint64_t *>(smem);  // [kStages] TMA landed          (count 1 + tx)
    uint64_t *bar_ready = bar_tma + kStages;                 // [kStages] stage post-processed (count 1)
    uint64_t *bar_empty = bar_ready + kStages;               // [kStages] consumers done       (count kConsumerWarps)
    int *tile_ctl = reinterpret_cast<int *>(smem + 96);      // quiet launch: last-CTA flag, first / last sharing CTA
    long long *prefix = reinterpret_cast<long long *>(smem + kPrefixOff);  // active launch: first item of every star
    float *cst = reinterpret_cast<float *>(smem + kHeaderBytes);    // active launch only: contrast of the current kind, [kR][kConsumers]
    unsigned char *stage0 = smem + kHeaderBytes + (ACTIVE ? kFinBytes : 0);

    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&bar_tma[s], 1);
            mbar_init(&bar_ready[s], 1);
            mbar_init(&bar_empty[s], kConsumerWarps);
        }
        fence_mbar_init();
        reinterpret_cast<ItemQueue *>(smem + 128)->tail = 0;
    }
    // (launched with programmatic stream serialization: everything above overlaps the predecessor's tail)
    trigger_dependents();
    grid_dependency_wait();
    if (ACTIVE) {
        for (int k = tid; k <= p.n_stars; k += kThreads)
            prefix[k] = k < p.n_stars ? (p.many ? __ldcg(&p.many[k].item0) : 0LL) : p.n_items;
    }
    __syncthreads();

    if (warp >= kConsumerWarps) {
        // =============================== producer warps ==============================================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsProducer));
        const int st = warp - kConsumerWarps;  // this warp's stage
        unsigned char *sb = stage0 + (size_t)st * p.stage_bytes;
        float *rs = reinterpret_cast<float *>(sb);
        const float2 *raw = reinterpret_cast<const float2 *>(sb + p.raw_off);
        float2 *rec = reinterpret_cast<float2 *>(sb + p.rec_off);
        int2 *runs = reinterpret_cast<int2 *>(sb + p.run_off);
        Desc *desc = reinterpret_cast<Desc *>(sb + p.desc_off);
        typename std::conditional<ACTIVE, ActiveSource, QuietSource>::type src;
        init_source(src, p, reinterpret_cast<ItemQueue *>(smem + 128), prefix,
                    reinterpret_cast<StarBlock *>(smem + kBlockCacheOff + (size_t)st * kBlockCacheStride), st == 0, smem + kOrderOff);
        Job jb;
        for (int n = st, use = 0;; n += kStages, ++use) {
            const int status = src.get(n, jb);
            if (status == kSrcBeyond) break;
            mbar_wait_backoff(&bar_empty[st], (uint32_t)((use & 1) ^ 1));
            if (status == kSrcExit) {
                if (lane == 0) {
                    desc->flags = kJobExit;
                    mbar_arrive(&bar_ready[st]);
                }
                break;
            }
            const StarBlock &blk = source_block(src, p);  // quiet: the kernel argument; active: this warp's cached copy
            const int H = blk.halo;
            const int span = span_px(H);
            const long long row_len = blk.row_len, n_pix = blk.n_pix;
            const double c0 = blk.c0;
            const long long m_t0 = jb.tile * kTile;
            const long long s_start = m_t0 - H;  // global pixel of smem position 0 (multiple of 4)
            if (lane == 0) {
                if (jb.count > 0) {
                    const long long g_lo = s_start < 0 ? 0 : s_start;
                    const long long g_hi = (s_start + span) < row_len ? (s_start + span) : row_len;
                    const uint32_t row_bytes = (uint32_t)((g_hi - g_lo) * (long long)sizeof(float));
                    const float *src_row = blk.base[EFFECTS ? (p.eff[jb.kind] & 3) : jb.kind] + (long long)jb.row * blk.pitch + g_lo;
                    const uint32_t ent_bytes = (uint32_t)(((jb.count + 1) & ~1) * (int)sizeof(float2));
                    fence_proxy_async_smem();
                    mbar_arrive_expect_tx(&bar_tma[st], row_bytes + ent_bytes);
                    tma_load_1d(sb + (size_t)(g_lo - s_start) * sizeof(float), src_row, row_bytes, &bar_tma[st]);
                    tma_load_1d(sb + p.raw_off, blk.ent + jb.begin, ent_bytes, &bar_tma[st]);
                } else {
                    mbar_arrive(&bar_tma[st]);  // nothing to load: keeps the barrier's phase in step
                }
            }
            mbar_wait(&bar_tma[st], (uint32_t)(use & 1));
            // -- records, run table, edge halo, descriptor ---------------------------------------------
            const float c_first = (float)(c0 + (double)m_t0);
            const float c_last = (float)(c0 + (double)(m_t0 + kTile - 1));
            const int n_runs = build_runs(raw, jb.count, c_first, c_last, H, p.collapse, rec, runs);
            if (lane == 0) {
                runs[n_runs] = make_int2(p.collapse ? n_runs : jb.count, 0);  // sentinel: end of the last run
                desc->m_t0 = m_t0;
                desc->flags = jb.flags;
                desc->kind = jb.kind;
                desc->out_idx = jb.out_idx;
                desc->n_runs = n_runs;
                desc->star = jb.star;
                desc->halo = H;
                desc->c0 = c0;
                desc->out_lo = blk.out_lo;
                desc->out_hi = blk.out_hi;
                desc->out_pitch = blk.out_pitch;
                desc->out = blk.out;
                if (EFFECTS) {
                    desc->out_fc[0] = blk.out_fc[0];
                    desc->out_fc[1] = blk.out_fc[1];
                }
                desc->contrast[0] = blk.contrast[1];
                desc->contrast[1] = blk.contrast[2];
            }
            if (jb.count > 0) {
                if (s_start < 0) {  // clamp-to-edge below the grid (reading S8)
                    const int nb = (int)(-s_start);
                    const float v = rs[nb];
                    for (int q = lane; q < nb; q += 32) rs[q] = v;
                }
                if (s_start + span > n_pix) {  // ... and above it
                    const int first = (int)(n_pix - s_start);
                    const float v = rs[first - 1];
                    for (int q = first + lane; q < span; q += 32) rs[q] = v;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_ready[st]);
        }
        return;
    }

    // =================================== consumer warps ===============================================
    if (EFFECTS) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsConsumerEffects));
    else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsConsumer));
    int H = p.halo, base0 = H + tid;  // halo of the current item's star; smem position of pixel r = 0 at zero shift
    int cmask = 0;                     // bit k: kind k of the current item's star carries a contrast array
    long long out_lo = 0, out_hi = 0;  // of the current item's star
    long long m_t0 = 0;
    float cmf = 0.f;      // lambda0/k + m of this thread's first pixel
    // W lerp = W (s + t d), t = a c - q  ==>  W u + c (W a) d  with u = s - q d: the per-pixel factor c = lambda0/k + m is
    // pulled out of the sum over entries.  acc1 collects W u, acc2 collects (W a) d; pair k = pixels r = 2k, 2k + 1 (the
    // operands of one packed FMA).  A fold adds acc1 + c acc2 to the fp64 totals.
    float2 acc1[kR / 2], acc2[kR / 2];
    double tot[NOUT][kR];
    int cnt = 0, cur_kind = 0;
    int kcode = 0;  // effects launch: Params::eff of the current kind
    // a6: post-shift contrast (I_ratio of Eq. 3) per output pixel: a fold multiplies the fp32 partial sums of the current
    // kind by the kind's contrast C[m] in fp64 (the product is exact) on their way into the fp64 totals - no per-kind
    // totals are kept.  The contrast values of the current kind are fetched with cp.async while its first jobs run.
    int rmax = 0;            // pixels r < rmax of this thread lie inside the spectrum
    bool kind_c = false;     // the current kind carries a contrast array
    const Desc *desc = nullptr;  // descriptor of the current job
    auto fold = [&]() {
        if (EFFECTS) {
            // (a + b C) P per output: a, b from the kind's code; C = 1 where the kind carries no contrast array
            if (kind_c) cp_async_wait_all();
            double ma[NOUT], mb[NOUT];
#pragma unroll
            for (int o = 0; o < NOUT; ++o) {
                const int c = (kcode >> (4 + 2 * o)) & 3;
                ma[o] = (c == kMulOne || c == kMulOneMinusC) ? 1.0 : 0.0;
                mb[o] = c == kMulC ? 1.0 : c == kMulOneMinusC ? -1.0 : 0.0;
            }
#pragma unroll
            for (int k = 0; k < kR / 2; ++k) {
                const float c0 = cmf + (float)(kConsumers * 2 * k), c1 = cmf + (float)(kConsumers * (2 * k + 1));
                const double w0 = (kind_c && 2 * k < rmax) ? (double)cst[(2 * k) * kConsumers + tid] : 1.0;
                const double w1 = (kind_c && 2 * k + 1 < rmax) ? (double)cst[(2 * k + 1) * kConsumers + tid] : 1.0;
                const double p0 = (double)fmaf(c0, acc2[k].x, acc1[k].x), p1 = (double)fmaf(c1, acc2[k].y, acc1[k].y);
#pragma unroll
                for (int o = 0; o < NOUT; ++o) {
                    tot[o][2 * k] = fma(p0, fma(mb[o], w0, ma[o]), tot[o][2 * k]);
                    tot[o][2 * k + 1] = fma(p1, fma(mb[o], w1, ma[o]), tot[o][2 * k + 1]);
                }
                acc1[k] = make_float2(0.f, 0.f);
                acc2[k] = make_float2(0.f, 0.f);
            }
        } else if (ACTIVE && kind_c) {
            cp_async_wait_all();
#pragma unroll
            for (int k = 0; k < kR / 2; ++k) {
                const float c0 = cmf + (float)(kConsumers * 2 * k), c1 = cmf + (float)(kConsumers * (2 * k + 1));
                const double w0 = 2 * k < rmax ? (double)cst[(2 * k) * kConsumers + tid] : 1.0;
                const double w1 = 2 * k + 1 < rmax ? (double)cst[(2 * k + 1) * kConsumers + tid] : 1.0;
                tot[0][2 * k] = fma((double)fmaf(c0, acc2[k].x, acc1[k].x), w0, tot[0][2 * k]);
                tot[0][2 * k + 1] = fma((double)fmaf(c1, acc2[k].y, acc1[k].y), w1, tot[0][2 * k + 1]);
                acc1[k] = make_float2(0.f, 0.f);
                acc2[k] = make_float2(0.f, 0.f);
            }
        } else {
#pragma unroll
            for (int k = 0; k < kR / 2; ++k) {
                const float c0 = cmf + (float)(kConsumers * 2 * k), c1 = cmf + (float)(kConsumers * (2 * k + 1));
                tot[0][2 * k] += (double)fmaf(c0, acc2[k].x, acc1[k].x);
                tot[0][2 * k + 1] += (double)fmaf(c1, acc2[k].y, acc1[k].y);
                acc1[k] = make_float2(0.f, 0.f);
                acc2[k] = make_float2(0.f, 0.f);
            }
        }
        cnt = 0;
    };
    auto begin_kind = [&](int kind) {  // after a fold: only this thread ever touches its 16 slots of `cst`
        cur_kind = kind;
        int ctype = kind;  // region type whose contrast array the kind's partial sums meet
        if (EFFECTS) {
            kcode = p.eff[kind];
            ctype = (kcode >> 2) & 3;
        }
        kind_c = (cmask >> ctype) & 1;
        if (!kind_c) return;
        const float *ck = desc->contrast[ctype - 1];
#pragma unroll
        for (int r = 0; r < kR; ++r)
            if (r < rmax) cp_async_4(&cst[r * kConsumers + tid], ck + m_t0 + tid + kConsumers * r);
        cp_async_commit();
    };

    for (int n = 0;; ++n) {
        const int st = n % kStages;
        mbar_wait(&bar_ready[st], (uint32_t)((n / kStages) & 1));
        const unsigned char *sb = stage0 + (size_t)st * p.stage_bytes;
        const float *rs = reinterpret_cast<const float *>(sb);
        const float2 *raw = reinterpret_cast<const float2 *>(sb + p.raw_off);
        const float2 *rec = reinterpret_cast<const float2 *>(sb + p.rec_off);
        const int2 *runs = reinterpret_cast<const int2 *>(sb + p.run_off);
        desc = reinterpret_cast<const Desc *>(sb + p.desc_off);
        const int flags = desc->flags;
        if (flags & kJobExit) break;
        const int n_runs = desc->n_runs;
        const int kind = desc->kind;
        const int out_idx = desc->out_idx;
        if (flags & kJobFirst) {
            m_t0 = desc->m_t0;
            H = desc->halo;
            base0 = H + tid;
            out_lo = desc->out_lo;
            out_hi = desc->out_hi;
            cmask = (desc->contrast[0] ? 2 : 0) | (desc->contrast[1] ? 4 : 0);
            cmf = (float)(desc->c0 + (double)(m_t0 + tid));
#pragma unroll
            for (int r = 0; r < kR; ++r)
#pragma unroll
                for (int o = 0; o < NOUT; ++o) tot[o][r] = 0.0;
#pragma unroll
            for (int k = 0; k < kR / 2; ++k) acc1[k] = acc2[k] = make_float2(0.f, 0.f);
            cnt = 0;
            if (ACTIVE) {
                const long long rem = out_hi - (m_t0 + tid);
                rmax = rem <= 0 ? 0 : (int)min((long long)kR, (rem + kConsumers - 1) / kConsumers);
                begin_kind(kind);
            }
        }
        if (ACTIVE && kind != cur_kind) {
            // the multiplier changes: what was summed so far goes to the totals
            if (EFFECTS || kind_c || ((cmask >> kind) & 1)) fold();
            begin_kind(kind);
        }
        int2 run_next = runs[0];
        for (int ri = 0; ri < n_runs; ++ri) {
            const int2 run = run_next;
            run_next = runs[ri + 1];  // the next run's header is fetched while this run is processed
            const int nxt = run_next.x;
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
                    float &ar = (r & 1) ? acc1[r / 2].y : acc1[r / 2].x;
                    ar = fmaf(en.y, fmaf(t, s1 - s0, s0), ar);
                }
                if (++cnt >= kFold) fold();
                continue;
            }
            // u = s - q d and d = s[+1] - s are per-pixel registers of the run
            float2 u[kR / 2], v[kR / 2];
            {
                const float *wv = rs + base0 + run.y;
                const float2 nq = bcast2(-(float)run.y);
#pragma unroll
                for (int k = 0; k < kR / 2; ++k) {
                    const float2 s0 = make_float2(wv[kConsumers * 2 * k], wv[kConsumers * (2 * k + 1)]);
                    const float2 s1 = make_float2(wv[kConsumers * 2 * k + 1], wv[kConsumers * (2 * k + 1) + 1]);
                    v[k] = fma2(bcast2(-1.f), s0, s1);
                    u[k] = fma2(nq, v[k], s0);
                }
            }
            const int len = p.collapse ? 1 : nxt - run.x;
            const float2 *re = rec + run.x;
            float2 rc = re[0];  // {W, W a}; the next record is fetched while this one is used
#pragma unroll 2
            for (int i = 0; i < len; ++i) {
                const float2 nx = re[i + 1];  // one past the run's end is still inside the stage
#pragma unroll
                for (int k = 0; k < kR / 2; ++k) acc1[k] = fma2(bcast2(rc.x), u[k], acc1[k]);  // (1) + W u_r
#pragma unroll
                for (int k = 0; k < kR / 2; ++k) acc2[k] = fma2(bcast2(rc.y), v[k], acc2[k]);  // (2) + (W a) d_r
                rc = nx;
            }
            cnt += len;
            if (cnt >= kFold) fold();  // at most kFold + one run's entries are ever summed in fp32
        }
        float *o_row = nullptr;  // active launch: this thread's first output pixel (read before the stage is released)
        float *o_fc[2] = {nullptr, nullptr};
        if (ACTIVE && (flags & kJobLast)) {
            const long long off = (long long)out_idx * desc->out_pitch + m_t0 + tid;
            o_row = (EFFECTS && !desc->out) ? nullptr : desc->out + off;
            if (EFFECTS) {
                o_fc[0] = desc->out_fc[0] ? desc->out_fc[0] + off : nullptr;
                o_fc[1] = desc->out_fc[1] ? desc->out_fc[1] + off : nullptr;
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar_empty[st]);  // the stage may be refilled while the tile is stored

        if (flags & kJobLast) {
            fold();
            if (ACTIVE) {
#pragma unroll
                for (int oi = 0; oi < NOUT; ++oi) {
                    float *o = oi == 0 ? o_row : o_fc[oi - 1];
                    if (EFFECTS && !o) continue;
#pragma unroll
                    for (int r = 0; r < kR; ++r)
                        if (r < rmax && m_t0 + tid + kConsumers * r >= out_lo) o[kConsumers * r] = (float)tot[oi][r];
                }
            } else {
                double *o = p.partial + ((long long)blockIdx.x * p.max_seg + out_idx) * kTile;
#pragma unroll
                for (int r = 0; r < kR; ++r) o[tid + kConsumers * r] = tot[0][r];
                // a6: the last CTA to deliver its share of this tile adds all shares in CTA order (the same
                // order whoever comes last: deterministic) and rounds once to fp32.
                const long long tile = m_t0 / kTile;
                const long long E = __ldcg(&p.row_start[p.one.n_mu]), U = E * p.one.n_tiles, G = gridDim.x;
                const long long ub = tile * E, ue = ub + E;
                __threadfence();
                consumer_bar_sync();
                if (tid == 0) {
                    long long c = (ub * G) / U;
                    while (c > 0 && range_begin(c, U, G) > ub) --c;
                    while (c + 1 < G && range_begin(c + 1, U, G) <= ub) ++c;
                    int n = 0;
                    long long c_lo = c, c_hi = c;
                    for (; c < G; ++c) {
                        const long long b = range_begin(c, U, G), e = range_begin(c + 1, U, G);
                        if (b >= ue) break;
                        if (e <= b || e <= ub) continue;
                        c_hi = c;
                        ++n;
                    }
                    const int ticket = atomicAdd(&p.tile_ticket[tile], 1);
                    const bool last = ticket == n - 1;
                    if (last) p.tile_ticket[tile] = 0;  // ready for the next launch
                    tile_ctl[0] = last ? 1 : 0;
                    tile_ctl[1] = (int)c_lo;
                    tile_ctl[2] = (int)c_hi;
                }
                consumer_bar_sync();
                if (tile_ctl[0]) {
                    __threadfence();
                    double sum[kR];
#pragma unroll
                    for (int r = 0; r < kR; ++r) sum[r] = 0.0;
                    for (long long c = tile_ctl[1]; c <= tile_ctl[2]; ++c) {
                        const long long b = range_begin(c, U, G), e = range_begin(c + 1, U, G);
                        if (e <= b || e <= ub) continue;
                        const double *src = p.partial + ((c * p.max_seg + (tile - b / E)) * kTile) + tid;
#pragma unroll
                        for (int r = 0; r < kR; ++r) sum[r] += __ldcg(&src[kConsumers * r]);
                    }
                    float *qo = p.one.out + m_t0 + tid;
#pragma unroll
                    for (int r = 0; r < kR; ++r)
                        if (m_t0 + tid + kConsumers * r < out_hi && m_t0 + tid + kConsumers * r >= out_lo)
                            qo[kConsumers * r] = (float)sum[r];
                }
                consumer_bar_sync();  // tile_ctl may be rewritten by the next tile
            }
        }
    }
}

}  // namespace f32
}  // namespace soap
