// Host side of the C ABI declared in include/soap_b200.h: argument checks, scratch management and
// kernel launches.  Every step of the path runs in the kernels of geometry.cuh / active.cuh / sia.cuh;
// nothing here computes spectra on the CPU.  The only host arithmetic is O(n_regions * n_phases) region
// centres (Localize of PAPER.md:69-71) and halo / grid sizing from the star parameters.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <type_traits>
#include <utility>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/soap_b200.h"
#include "active.cuh"
#include "composite.cuh"
#include "contrast.cuh"
#include "geometry.cuh"
#include "lsf.cuh"
#include "rv.cuh"
#include "sia.cuh"
#include "sia_f32.cuh"

namespace {

using namespace soap;

std::string g_create_error;

template <typename T>
struct DevBuf {
    T *ptr = nullptr;
    size_t cap = 0;  // elements
    cudaError_t reserve(size_t n) {
        if (n <= cap) return cudaSuccess;
        if (ptr) cudaFree(ptr);
        ptr = nullptr;
        cap = 0;
        cudaError_t e = cudaMalloc(reinterpret_cast<void **>(&ptr), n * sizeof(T));
        if (e == cudaSuccess) cap = n;
        return e;
    }
    void release() {
        if (ptr) cudaFree(ptr);
        ptr = nullptr;
        cap = 0;
    }
};

}  // namespace

struct soap_star {
    int device = 0;
    int n_sm = 148;
    std::string err;
    bool ready = false;

    // star
    soap_star_params prm{};
    std::vector<double> mu_centres;
    double sini = 1.0, cosi = 0.0;
    double amax = 0.0;  // host bound on max |D - 1|
    int form = SOAP_FORM_AUTO, form_used = SOAP_FORM_BINNED;
    long long out_lo_override = -1, out_hi_override = -1;  // soap_synthesize_host: pixels of a window that are stored
    long long clip_override = 0;    // soap_synthesize_host: readable row length of a window into a wider table (0 = pitch)
    int lists_kinds = 3;            // kinds of the entry lists the last active map wrote (effect_kinds)
    bool reuse_lists = false;       // soap_synthesize_host: the active map of the previous call is still valid
    bool regions_uploaded = false;  // soap_synthesize_host: the region centres are already on the device
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    std::vector<cudaEvent_t> ev_pipe;
    long long active_pool_cap = 0;  // per-cell active form: entries one phase's pool must hold (from the region radii)
    bool cell_entries = false;  // one entry per cell (SOAP_FORM_CELLS, or differential rotation) instead of per (column, mu-bin)
    int opt_quiet_splits = 0;
    bool opt_timing = false;
    bool opt_effect_passes = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};  // quiet start/stop, active start/stop
    bool ev_valid[2] = {false, false};

    // geometry (device)
    DevBuf<double> d_mu, d_w, d_vel, d_col_a, d_Wbin, d_col_sumw;
    DevBuf<int> d_bin, d_col_nvis, d_row_start, d_colcnt, d_cellpos;
    DevBuf<float2> d_ent32;
    DevBuf<double2> d_ent64;
    DevBuf<DevInfo> d_info;
    DevBuf<unsigned int> d_geom_done;
    size_t ent_cap = 0;
    // composite-column form: pair tables built by the geometry kernel
    DevBuf<float2> d_cWp;
    DevBuf<comp::PairHdr> d_chdr;
    int comp_stride = 0;  // bins per table row (multiple of 4); 0 = tables not built
    DevBuf<comp::Star> d_cstars;
    DevBuf<unsigned char> d_gargs;  // batch geometry: the stars' kernel arguments (owned by the first star of the batch)  // batch launches: the stars' descriptors (owned by the first star of the batch)

    // quiet scratch
    DevBuf<double> d_partial;
    DevBuf<int> d_tile_ticket;

    // active scratch
    DevBuf<RegionAtPhase> d_rp;
    struct PinnedSlot {  // ring of pinned staging buffers: a slot is reused only after its copy completed
        RegionAtPhase *ptr = nullptr;
        size_t cap = 0;
        cudaEvent_t done = nullptr;
        bool in_flight = false;
    } h_rp[4];
    int h_rp_next = 0;
    DevBuf<unsigned char> d_aent;
    DevBuf<int> d_segcnt, d_nactive, d_sched;
    DevBuf<ActiveJob> d_jobs;
    DevBuf<ActiveCounters> d_counters;
    // f32 active launch: region centres + map arguments + star blocks of a call (a batch: of all its stars), staged in one
    // pinned buffer and copied with one cudaMemcpyAsync (owned by the first star of the batch)
    DevBuf<unsigned char> d_call;
    struct PinnedBytes {
        unsigned char *ptr = nullptr;
        size_t cap = 0;
        cudaEvent_t done = nullptr;
        bool in_flight = false;
    } h_call[4];
    int h_call_next = 0;
    size_t call_rp_off = 0, call_prep_off = 0, call_blk_off = 0, call_ph_off = 0;  // sections of d_call of the last prepared call
    bool attr_active_set = false, attr_geom_set = false, attr_rv_set = false;
    bool attr_prep_set[4] = {false, false, false, false};  // active_prepare_kernel per (threads, inline regions)
    int occ_active = 0, occ_effects = 0;
    size_t occ_active_smem = 0, occ_effects_smem = 0;
    bool attr_effects_set = false;

    // host-buffer staging (soap_synthesize_host)
    DevBuf<unsigned char> d_stage[3], d_stage_c[3], d_out_q, d_out_d;

    // stats
    int last_quiet_splits = 0, last_tile_px = 0, launches = 0, last_form = 0;
    long long last_active_cells = 0;
    int last_n_phases = 0;  // phases of the last active call: d_sched = [n_jobs | entries] of each

    int fail(int code, const char *fmt, ...) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof(buf), fmt, ap);
        va_end(ap);
        err = buf;
        return code;
    }
};

namespace {

#define SOAP_CUDA(star, call)                                                                            \
    do {                                                                                                 \
        cudaError_t e__ = (call);                                                                        \
        if (e__ != cudaSuccess)                                                                          \
            return (star)->fail(e__ == cudaErrorMemoryAllocation ? SOAP_ERR_OOM : SOAP_ERR_CUDA,         \
                                "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

#define SOAP_LAUNCH_CHECK(star, name)                                                                    \
    do {                                                                                                 \
        cudaError_t e__ = cudaGetLastError();                                                            \
        if (e__ != cudaSuccess)                                                                          \
            return (star)->fail(SOAP_ERR_CUDA, "launch of %s failed: %s", name, cudaGetErrorString(e__)); \
        (star)->launches++;                                                                              \
    } while (0)

// Launch with programmatic stream serialization: the kernel may be scheduled while its predecessor in the stream drains;
// it calls grid_dependency_wait() (ptx_helpers.cuh) before it reads what the predecessor wrote.  The four launches of a
// step (geometry, quiet, active map, active delta) are chained this way: launch latency and prologues overlap the tails.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

inline double host_dshift(double v_kms, int mode) {
    const double b = v_kms / kSpeedOfLightKms;
    if (mode == 1) return -b;
    return -2.0 * b / ((1.0 + b) + std::sqrt(1.0 - b * b));
}

inline int round_up4(long long v) { return (int)((v + 3) & ~3LL); }
inline bool n_mu_ok_for_composite(int n_mu) { return n_mu >= 1 && n_mu <= comp::kMaxBins; }

int check_spectra(soap_star *s, const soap_spectra *sp, const char *name) {
    if (!sp) return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: NULL", name);
    if (!sp->data) return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: data is NULL", name);
    if (sp->n_pix < 2) return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: n_pix must be >= 2", name);
    if (sp->n_pix > (1LL << 30)) return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: n_pix too large", name);
    if (sp->pitch < sp->n_pix || (sp->pitch & 3))
        return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: pitch must be >= n_pix and a multiple of 4", name);
    if (sp->dtype != SOAP_F32 && sp->dtype != SOAP_F64)
        return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: unknown dtype %d", name, sp->dtype);
    if (reinterpret_cast<uintptr_t>(sp->data) & 15)
        return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: data must be 16-byte aligned", name);
    if (!(sp->dlambda > 0.0) || !(sp->lambda0 > 0.0) || !std::isfinite(sp->dlambda) || !std::isfinite(sp->lambda0))
        return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: lambda0 and dlambda must be positive and finite", name);
    if (!std::isfinite(sp->lb_c0) || !std::isfinite(sp->lb_c1) || !std::isfinite(sp->lb_c2))
        return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: limb-brightening coefficients must be finite", name);
    return SOAP_OK;
}

int check_same_grid(soap_star *s, const soap_spectra *a, const soap_spectra *b, const char *name) {
    if (a->n_pix != b->n_pix || a->dtype != b->dtype || a->lambda0 != b->lambda0 || a->dlambda != b->dlambda)
        return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: n_pix / dtype / lambda0 / dlambda differ from quiet", name);
    if (a->pitch != b->pitch) return s->fail(SOAP_ERR_INVALID_ARG, "%s spectra: pitch differs from quiet", name);
    return SOAP_OK;
}

int halo_for(const soap_star *s, const soap_spectra *sp) {
    const double c0 = sp->lambda0 / sp->dlambda;
    const double maxd = s->amax * (c0 + (double)sp->n_pix) * (1.0 + 1e-6);
    return round_up4((long long)std::ceil(maxd) + 2);
}

template <typename T, bool ACTIVE>
int launch_sia(soap_star *s, const SiaParams<T> &p, dim3 grid, cudaStream_t st) {
    const size_t smem = sia_smem_bytes<T>(p.halo);
    if (smem > 227 * 1024) return s->fail(SOAP_ERR_UNSUPPORTED, "shift of %d pixels needs %zu B of shared memory", p.halo, smem);
    static bool attr_set[64] = {};  // once per device and instantiation: the limit, not the launch's size (that is checked above)
    if (!attr_set[s->device & 63]) {
        SOAP_CUDA(s, cudaFuncSetAttribute(sia_kernel<T, ACTIVE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        attr_set[s->device & 63] = true;
    }
    const int e0 = ACTIVE ? 2 : 0;
    if (s->opt_timing) {
        for (int k = e0; k < e0 + 2; ++k)
            if (!s->ev[k]) SOAP_CUDA(s, cudaEventCreate(&s->ev[k]));
        SOAP_CUDA(s, cudaEventRecord(s->ev[e0], st));
    }
    sia_kernel<T, ACTIVE><<<grid, kThreads, smem, st>>>(p);
    SOAP_LAUNCH_CHECK(s, ACTIVE ? "sia_kernel<active>" : "sia_kernel<quiet>");
    if (s->opt_timing) {
        SOAP_CUDA(s, cudaEventRecord(s->ev[e0 + 1], st));
        s->ev_valid[ACTIVE ? 1 : 0] = true;
    }
    return SOAP_OK;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize of f32::sia_f32_kernel<ACTIVE>, set once per device to the limit every launch
// is checked against (the attribute is a ceiling: occupancy follows the launch's own size)
template <bool ACTIVE>
int sia_f32_attr(soap_star *s) {
    static bool attr_set[64] = {};
    if (!attr_set[s->device & 63]) {
        SOAP_CUDA(s, cudaFuncSetAttribute(f32::sia_f32_kernel<ACTIVE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        attr_set[s->device & 63] = true;
    }
    return SOAP_OK;
}

// fp32 spectra: warp-specialised kernel of sia_f32.cuh.  `which`: 0 = quiet, 1 = active (event slots).
template <bool ACTIVE>
int launch_sia_f32(soap_star *s, const f32::Params &p, dim3 grid, cudaStream_t st) {
    const size_t smem = f32::smem_bytes(p.halo, ACTIVE);
    if (smem > 227 * 1024) return s->fail(SOAP_ERR_UNSUPPORTED, "shift of %d pixels needs %zu B of shared memory", p.halo, smem);
    if (int rc = sia_f32_attr<ACTIVE>(s)) return rc;
    const int e0 = ACTIVE ? 2 : 0;
    if (s->opt_timing) {
        for (int k = e0; k < e0 + 2; ++k)
            if (!s->ev[k]) SOAP_CUDA(s, cudaEventCreate(&s->ev[k]));
        SOAP_CUDA(s, cudaEventRecord(s->ev[e0], st));
    }
    SOAP_CUDA(s, launch_pdl(f32::sia_f32_kernel<ACTIVE>, grid, dim3(f32::kThreads), smem, st, p));
    SOAP_LAUNCH_CHECK(s, ACTIVE ? "sia_f32_kernel<active>" : "sia_f32_kernel<quiet>");
    if (s->opt_timing) {
        SOAP_CUDA(s, cudaEventRecord(s->ev[e0 + 1], st));
        s->ev_valid[ACTIVE ? 1 : 0] = true;
    }
    return SOAP_OK;
}

int quiet_f32(soap_star *s, const soap_spectra *q, void *out, cudaStream_t st) {
    const long long P = q->n_pix;
    const int n_tiles = (int)((P + f32::kTile - 1) / f32::kTile);
    f32::Params p{};
    p.one.base[0] = static_cast<const float *>(q->data);
    p.one.pitch = q->pitch;
    p.one.row_len = s->clip_override > 0 ? s->clip_override : q->pitch;
    p.one.out_lo = s->out_lo_override >= 0 ? s->out_lo_override : 0;
    p.one.out_hi = s->out_hi_override >= 0 ? s->out_hi_override : P;
    p.one.n_pix = P;
    p.one.c0 = q->lambda0 / q->dlambda;
    p.one.n_mu = s->prm.n_mu;
    p.one.halo = halo_for(s, q);
    p.one.ent = s->d_ent32.ptr;
    p.one.n_tiles = n_tiles;
    p.n_stars = 1;
    p.halo = p.one.halo;
    f32::set_layout(p);
    p.collapse = s->form_used == SOAP_FORM_FIR ? 1 : 0;
    p.row_start = s->d_row_start.ptr;
    // one CTA per resident slot (a single wave); fewer when there is too little work to share out
    const size_t smem = f32::smem_bytes(p.halo, false);
    if (smem > 227 * 1024) return s->fail(SOAP_ERR_UNSUPPORTED, "shift of %d pixels needs %zu B of shared memory", p.halo, smem);
    if (int rc = sia_f32_attr<false>(s)) return rc;
    int occ = 0;
    SOAP_CUDA(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f32::sia_f32_kernel<false>, f32::kThreads, smem));
    if (occ < 1) return s->fail(SOAP_ERR_UNSUPPORTED, "quiet kernel does not fit on an SM (halo %d)", p.halo);
    long long G = s->opt_quiet_splits > 0 ? (long long)s->opt_quiet_splits : (long long)s->n_sm * occ;
    const long long max_entries = (long long)s->prm.grid_n * (s->cell_entries ? s->prm.grid_n : s->prm.n_mu);
    G = std::max(1LL, std::min(G, (long long)n_tiles * max_entries / 64));
    if (s->opt_quiet_splits <= 0) G = std::min(G, (long long)n_tiles * 8);  // few tiles: at most 8 CTAs share one (cheap hand-over)
    p.max_seg = (int)(n_tiles / G) + 3;
    SOAP_CUDA(s, s->d_partial.reserve((size_t)G * p.max_seg * f32::kTile));
    p.partial = s->d_partial.ptr;
    if ((size_t)n_tiles > s->d_tile_ticket.cap) {
        SOAP_CUDA(s, s->d_tile_ticket.reserve((size_t)n_tiles));
        SOAP_CUDA(s, cudaMemsetAsync(s->d_tile_ticket.ptr, 0, s->d_tile_ticket.cap * sizeof(int), st));  // self-resetting after
    }
    p.tile_ticket = s->d_tile_ticket.ptr;
    p.one.out = static_cast<float *>(out);
    int rc = launch_sia_f32<false>(s, p, dim3((unsigned)G), st);
    if (rc) return rc;
    s->last_quiet_splits = (int)G;
    s->last_tile_px = f32::kTile;
    return SOAP_OK;
}

// Composite-column form (composite.cuh): does the launch apply to this star and these spectra?
bool composite_applies(const soap_star *s, const soap_spectra *q) {
    if (s->form_used != SOAP_FORM_COMPOSITE || s->comp_stride == 0 || q->dtype != SOAP_F32) return false;
    const int H = halo_for(s, q);
    if (2 * H > comp::kSpan / 2) return false;  // at most half of a span is halo
    const int n_pairs = (s->prm.grid_n + 1) / 2;
    return comp::smem_bytes(s->comp_stride, n_pairs, H) <= (size_t)200 * 1024 / comp::kCtasPerSm;
}

void composite_fill(const soap_star *s, const soap_spectra *q, void *out, comp::Star &c) {
    c.base = static_cast<const float *>(q->data);
    c.out = static_cast<float *>(out);
    c.Wp = s->d_cWp.ptr;
    c.hdr = s->d_chdr.ptr;
    c.ticket = s->d_tile_ticket.ptr;
    c.pitch = q->pitch;
    c.n_pix = q->n_pix;
    c.out_lo = s->out_lo_override >= 0 ? s->out_lo_override : 0;
    c.out_hi = s->out_hi_override >= 0 ? s->out_hi_override : q->n_pix;
    c.c0 = q->lambda0 / q->dlambda;
    c.n_mu = s->prm.n_mu;
    c.n_pairs = (s->prm.grid_n + 1) / 2;
    c.halo = halo_for(s, q);
    c.L = comp::kSpan - 2 * c.halo;
    c.n_tiles = (int)((q->n_pix + c.L - 1) / c.L);
    c.wp_stride = s->comp_stride;
}

template <int NB>
int launch_composite_nb(soap_star *s, const comp::Params &p, unsigned G, size_t smem, cudaStream_t st) {
    static bool attr_set[64] = {};
    if (!attr_set[s->device & 63]) {
        SOAP_CUDA(s, cudaFuncSetAttribute(comp::composite_quiet_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_set[s->device & 63] = true;
    }
    SOAP_CUDA(s, launch_pdl(comp::composite_quiet_kernel<NB>, dim3(G), dim3(comp::kThreads), smem, st, p));
    return SOAP_OK;
}

// One launch for n_stars stars (n_stars == 1: the descriptor travels as a kernel argument).  `owner` provides the
// scratch and the timing events.
int launch_composite(soap_star *owner, const comp::Star *host_stars, const comp::Star *dev_stars, int n_stars, int nb,
                     int max_pairs, int max_mu, cudaStream_t st) {
    comp::Params p{};
    p.one = host_stars[0];
    p.many = n_stars > 1 ? dev_stars : nullptr;
    p.n_stars = n_stars;
    p.max_pairs = max_pairs;
    int max_halo = 0;
    for (int k = 0; k < n_stars; ++k) max_halo = std::max(max_halo, host_stars[k].halo);
    p.plane = comp::plane_floats(max_halo);
    // every CTA's range must hold at least one whole pair of every tile it shares (composite.cuh, ticket count)
    const long long cmax = 8LL * ((max_mu + 1) / 2) + comp::kPairCostBase;
    long long min_units = 0;
    for (int k = 0; k < n_stars; ++k) min_units += (long long)host_stars[k].n_tiles * host_stars[k].n_pairs * comp::kPairCostBase;
    // (short spectra: a CTA's range should hold a few pairs of every tile it shares - the span loads and the hand-over of the
    // shares are what a small launch costs; C2: 60 - 80 CTAs 26.6 us, 40 or 86 CTAs 30.7 us)
    long long G = std::max(1LL, std::min((long long)owner->n_sm * comp::kCtasPerSm, min_units * 2 / (5 * cmax)));
    if (owner->opt_quiet_splits > 0) G = std::max(1LL, std::min(G, (long long)owner->opt_quiet_splits));  // SOAP_OPT_QUIET_SPLITS caps the grid
    SOAP_CUDA(owner, owner->d_partial.reserve((size_t)G * 2 * comp::kSpan));
    p.partial = owner->d_partial.ptr;
    const size_t smem = comp::smem_bytes(nb, max_pairs, max_halo);
    if (smem > (size_t)200 * 1024 / comp::kCtasPerSm) return owner->fail(SOAP_ERR_UNSUPPORTED, "composite launch needs %zu B of shared memory", smem);
    if (owner->opt_timing) {
        for (int k = 0; k < 2; ++k)
            if (!owner->ev[k]) SOAP_CUDA(owner, cudaEventCreate(&owner->ev[k]));
        SOAP_CUDA(owner, cudaEventRecord(owner->ev[0], st));
    }
    int rc = SOAP_OK;
    switch (nb) {
        case 4: rc = launch_composite_nb<4>(owner, p, (unsigned)G, smem, st); break;
        case 8: rc = launch_composite_nb<8>(owner, p, (unsigned)G, smem, st); break;
        case 12: rc = launch_composite_nb<12>(owner, p, (unsigned)G, smem, st); break;
        case 16: rc = launch_composite_nb<16>(owner, p, (unsigned)G, smem, st); break;
        case 20: rc = launch_composite_nb<20>(owner, p, (unsigned)G, smem, st); break;
        default: rc = launch_composite_nb<24>(owner, p, (unsigned)G, smem, st); break;
    }
    if (rc) return rc;
    SOAP_LAUNCH_CHECK(owner, "composite_quiet_kernel");
    if (owner->opt_timing) {
        SOAP_CUDA(owner, cudaEventRecord(owner->ev[1], st));
        owner->ev_valid[0] = true;
    }
    owner->last_quiet_splits = (int)G;
    return SOAP_OK;
}

int reserve_tickets(soap_star *s, size_t n_tiles, cudaStream_t st) {
    if (n_tiles > s->d_tile_ticket.cap) {
        SOAP_CUDA(s, s->d_tile_ticket.reserve(n_tiles));
        SOAP_CUDA(s, cudaMemsetAsync(s->d_tile_ticket.ptr, 0, s->d_tile_ticket.cap * sizeof(int), st));  // self-resetting after
    }
    return SOAP_OK;
}

int quiet_composite(soap_star *s, const soap_spectra *q, void *out, cudaStream_t st) {
    comp::Star c{};
    composite_fill(s, q, out, c);
    int rc = reserve_tickets(s, (size_t)c.n_tiles + 1, st);
    if (rc) return rc;
    c.ticket = s->d_tile_ticket.ptr;
    rc = launch_composite(s, &c, nullptr, 1, s->comp_stride, c.n_pairs, s->prm.n_mu, st);
    if (rc) return rc;
    s->last_tile_px = c.L;
    s->last_form = SOAP_FORM_COMPOSITE;
    return SOAP_OK;
}

template <typename T>
int quiet_impl(soap_star *s, const soap_spectra *q, void *out, cudaStream_t st) {
    if (sizeof(T) == 4 && composite_applies(s, q)) return quiet_composite(s, q, out, st);
    s->last_form = s->form_used == SOAP_FORM_COMPOSITE ? SOAP_FORM_BINNED : s->form_used;  // binned entries serve the rest
    if (sizeof(T) == 4) return quiet_f32(s, q, out, st);
    constexpr int TP = sia_tile_px<T>();
    const long long P = q->n_pix;
    const int n_tiles = (int)((P + TP - 1) / TP);
    int splits = s->opt_quiet_splits;
    if (splits <= 0) {
        // ~8 CTAs of 128 threads per SM; the entry list is cut into `splits` chunks per wavelength tile
        splits = (int)std::lround((double)(s->n_sm * 8) / n_tiles);
        const long long max_entries = (long long)s->prm.grid_n * (s->cell_entries ? s->prm.grid_n : s->prm.n_mu);
        const int cap = (int)std::max(1LL, max_entries / 16);
        splits = std::max(1, std::min(std::min(splits, 256), cap));
    }
    const long long part_pitch = (P + 3) & ~3LL;
    SOAP_CUDA(s, s->d_partial.reserve((size_t)splits * part_pitch));
    SiaParams<T> p{};
    p.base[0] = static_cast<const T *>(q->data);
    p.pitch = q->pitch;
    p.n_pix = P;
    p.c0 = q->lambda0 / q->dlambda;
    p.n_mu = s->prm.n_mu;
    p.halo = halo_for(s, q);
    if (sizeof(T) == 4) p.ent = reinterpret_cast<const typename SiaTraits<T>::Ent *>(s->d_ent32.ptr);
    else p.ent = reinterpret_cast<const typename SiaTraits<T>::Ent *>(s->d_ent64.ptr);
    p.row_start = s->d_row_start.ptr;
    p.n_splits = splits;
    p.partial = s->d_partial.ptr;
    p.part_pitch = part_pitch;
    int rc = launch_sia<T, false>(s, p, dim3(n_tiles, splits), st);
    if (rc) return rc;
    const int threads = 256;
    const long long quads = (P + 3) / 4;
    reduce_partials_kernel<T><<<(unsigned)((quads + threads - 1) / threads), threads, 0, st>>>(
        s->d_partial.ptr, part_pitch, splits, P, static_cast<T *>(out));
    SOAP_LAUNCH_CHECK(s, "reduce_partials_kernel");
    s->last_quiet_splits = splits;
    s->last_tile_px = TP;
    return SOAP_OK;
}

inline int per_cell_cap(const soap_star *s, int n_mu, int ncap, int n_kinds = 3) {  // jobs one phase's list can hold
    if (s->prm.diff_rot != 0.0) return 3 * n_mu + (int)(s->active_pool_cap / kActiveJobCap) + 2;
    return n_kinds * n_mu * ((ncap + kActiveJobCap - 1) / kActiveJobCap);
}

// Localize (readings S11-S13): region centres in the observer frame for every phase, written to
// out[n_phases][n_regions] (HOST).
void localize_regions(const soap_star *s, const soap_region *regions, int n_regions, const double *phases, int n_phases,
                      const double *radii, RegionAtPhase *out) {
    const double pi = 3.14159265358979323846;
    for (int p = 0; p < n_phases; ++p) {
        for (int r = 0; r < n_regions; ++r) {
            const soap_region &g = regions[r];
            const double lat = g.lat_deg * pi / 180.0;
            const double L = g.lon_deg * pi / 180.0 + 2.0 * pi * phases[p];
            const double sx = std::cos(lat) * std::sin(L), sy = std::sin(lat), sz = std::cos(lat) * std::cos(L);
            RegionAtPhase &o = out[(size_t)p * n_regions + r];
            o.xr = sx;
            o.yr = sy * s->sini - sz * s->cosi;
            o.zr = sy * s->cosi + sz * s->sini;
            const double rad = radii ? radii[(size_t)p * n_regions + r] : g.radius;
            const bool present = rad > 0.0;
            o.cos_alpha = present ? std::sqrt(1.0 - rad * rad) : 2.0;
            o.chord = present ? 2.0 * std::sin(0.5 * std::asin(rad)) : 0.0;
            o.type = (!present || o.zr < -rad - 1e-9) ? 0 : g.type;  // absent at this phase, or entirely on the far side
            o.pad = 0;
        }
    }
}

// ---- f32 spectra, solid-body rotation: the active path of one call - of ALL the stars of a batch call - in ONE active-map
// launch and ONE shift-interpolate-accumulate launch.  Region centres (Localize), the map kernel's arguments and the
// stars' blocks are staged in one pinned buffer of the first star and cross in one copy.
struct ActiveCall {  // one star's arguments
    soap_star *s;
    const soap_spectra *q, *spot, *fac;
    const soap_region *regions;
    int n_regions;
    const double *phases;
    int n_phases;
    const double *radii;  // nullable
    void *out;
    long long out_pitch;
    void *out_flux, *out_cb;  // kEffectAll only (each nullable, like out)
};
constexpr int kEffectAll = 3;  // internal: total, flux only and CB only from one pass (sia_f32.cuh, effects launch)

inline bool lb_is_one(const soap_spectra *t) { return !t || (t->lb_c0 == 1.0 && t->lb_c1 == 0.0 && t->lb_c2 == 0.0); }
// kinds of the entry lists (active.cuh): 3; effects form 4, or 8 when a limb-brightening law differs from 1
inline int effect_kinds(int effect, const soap_spectra *spot, const soap_spectra *fac) {
    return effect != kEffectAll ? 3 : (lb_is_one(spot) && lb_is_one(fac)) ? 4 : 8;
}

inline size_t align16(size_t v) { return (v + 15) & ~(size_t)15; }

// `external_map`: the entry lists were built by the caller (per-cell form under differential rotation): only the blocks
// are staged.  `map_only`: stop after the active map (soap_synthesize_host builds it before the table uploads are queued,
// so that no small copy of the chunk loop waits behind them in the copy engine).  A single star's block travels as a
// kernel argument: without `prepare` such a call copies nothing.
int active_f32_launch(const ActiveCall *calls, int n, int effect, bool prepare, bool external_map, cudaStream_t st,
                      bool map_only = false) {
    soap_star *own = calls[0].s;
    const bool use_lb = effect != SOAP_EFFECT_CB, use_contrast = effect != SOAP_EFFECT_CB;
    const bool quiet_rows = effect == SOAP_EFFECT_FLUX;
    const bool all_effects = effect == kEffectAll;
    if (all_effects && n != 1) return own->fail(SOAP_ERR_UNSUPPORTED, "the one-pass effects form takes one star per launch");
    const int n_kinds = effect_kinds(effect, calls[0].spot, calls[0].fac);
    // ---- per-star scratch, totals --------------------------------------------------------------------------------------
    size_t n_rp = 0;
    long long total_phases = 0, n_items = 0;
    int max_halo = 0;
    size_t prep_smem = 0;
    for (int k = 0; k < n; ++k) {
        const ActiveCall &c = calls[k];
        soap_star *s = c.s;
        const int N = s->prm.grid_n, n_mu = s->prm.n_mu;
        const int ncap = ((N + 1) & ~1) + 2;
        const long long n_seg = (long long)c.n_phases * n_kinds * n_mu;
        if (n_seg * ncap >= (1LL << 31)) return s->fail(SOAP_ERR_UNSUPPORTED, "n_phases * %d * n_mu * N too large for one call", n_kinds);
        SOAP_CUDA(s, s->d_aent.reserve((size_t)n_seg * ncap * sizeof(float2) + 64));
        SOAP_CUDA(s, s->d_segcnt.reserve((size_t)n_seg));
        SOAP_CUDA(s, s->d_nactive.reserve((size_t)c.n_phases));
        if (!s->d_counters.ptr) {
            SOAP_CUDA(s, s->d_counters.reserve(1));
            SOAP_CUDA(s, cudaMemsetAsync(s->d_counters.ptr, 0, sizeof(ActiveCounters), st));  // once per handle
        }
        SOAP_CUDA(s, s->d_jobs.reserve((size_t)c.n_phases * per_cell_cap(s, n_mu, ncap, n_kinds)));
        SOAP_CUDA(s, s->d_sched.reserve((size_t)2 * c.n_phases));
        if (!external_map) {  // (an external map was built by active_prepare_cells_kernel, with its own limit: active_impl)
            const int chunk_cols = std::max(32, (N + kPrepCluster - 1) / kPrepCluster);
            if (prep_smem_bytes(n_mu, chunk_cols, N, c.n_regions, n_kinds) > 200 * 1024)
                return s->fail(SOAP_ERR_UNSUPPORTED, "grid_n %d with %d mu bins exceeds the active-map kernel's shared memory", N, n_mu);
            prep_smem = std::max(prep_smem, prep_smem_bytes(n_mu, chunk_cols, N, c.n_regions, n_kinds));
        }
        s->last_n_phases = c.n_phases;
        n_rp += (size_t)c.n_regions * c.n_phases;
        total_phases += c.n_phases;
        max_halo = std::max(max_halo, halo_for(s, c.q));
        n_items += (long long)c.n_phases * ((c.q->n_pix + f32::kTile - 1) / f32::kTile);
    }
    if (total_phases * kPrepCluster >= (1LL << 31) || n_items >= (1LL << 31) - (1LL << 20))
        return own->fail(SOAP_ERR_UNSUPPORTED, "too many phases / (phase, tile) items for one launch");
    const size_t smem = f32::smem_bytes(max_halo, true);
    if (smem > 227 * 1024) return own->fail(SOAP_ERR_UNSUPPORTED, "shift of %d pixels needs %zu B of shared memory", max_halo, smem);
    own->lists_kinds = n_kinds;

    // ---- staging: [region centres][map arguments][star blocks][first phase of every star] -------------------------------
    size_t rp_off = 0, prep_off = 0, blk_off = 0, ph_off = 0, total = 0;
    if (external_map) {
        prepare = false;
        blk_off = 0;
        ph_off = align16((size_t)n * sizeof(f32::StarBlock));
        total = ph_off;
        own->call_blk_off = blk_off;
        own->call_ph_off = ph_off;
    } else if (prepare) {
        prep_off = align16(n_rp * sizeof(RegionAtPhase));
        blk_off = align16(prep_off + (size_t)n * sizeof(PrepArgs));
        ph_off = align16(blk_off + (size_t)n * sizeof(f32::StarBlock));
        total = ph_off + (size_t)(n + 1) * sizeof(int);
        own->call_rp_off = rp_off;
        own->call_prep_off = prep_off;
        own->call_blk_off = blk_off;
        own->call_ph_off = ph_off;
    } else {  // the lists of the previous (prepared) call of these stars are reused: only the blocks change
        blk_off = own->call_blk_off;
        ph_off = own->call_ph_off;
        total = ph_off;
        if (n > 1 && (!own->d_call.ptr || blk_off + (size_t)n * sizeof(f32::StarBlock) > ph_off))
            return own->fail(SOAP_ERR_NOT_READY, "no prepared active map to reuse");
    }
    // a single star's region centres travel as a kernel argument when they fit: such a call copies nothing
    const bool inline_rp = prepare && n == 1 && n_rp <= (size_t)kInlineRegions;
    const bool stage = (prepare && !inline_rp) || n > 1;  // a single star without a new map needs no copy either
    std::vector<unsigned char> unstaged;
    soap_star::PinnedBytes dummy;
    soap_star::PinnedBytes &slot = stage ? own->h_call[own->h_call_next] : dummy;
    if (stage) own->h_call_next = (own->h_call_next + 1) & 3;
    if (!stage) {
        unstaged.resize(total + 16);
        dummy.ptr = unstaged.data();
        dummy.cap = unstaged.size();
    }
    if (slot.in_flight) {
        SOAP_CUDA(own, cudaEventSynchronize(slot.done));
        slot.in_flight = false;
    }
    if (stage && !slot.done) SOAP_CUDA(own, cudaEventCreateWithFlags(&slot.done, cudaEventDisableTiming));
    if (total > slot.cap) {
        if (slot.ptr) cudaFreeHost(slot.ptr);
        slot.ptr = nullptr;
        slot.cap = 0;
        SOAP_CUDA(own, cudaMallocHost(reinterpret_cast<void **>(&slot.ptr), total + 4096));
        slot.cap = total + 4096;
    }
    if (stage && total > own->d_call.cap) {
        SOAP_CUDA(own, cudaDeviceSynchronize());  // growing frees the old buffer, which an earlier launch may still read
        SOAP_CUDA(own, own->d_call.reserve(total + 4096));
    }
    unsigned char *h = slot.ptr, *d = own->d_call.ptr;
    f32::StarBlock *hb = reinterpret_cast<f32::StarBlock *>(h + blk_off);
    PrepArgs *hp = reinterpret_cast<PrepArgs *>(h + prep_off);
    int *hph = reinterpret_cast<int *>(h + ph_off);
    size_t rp_pos = 0;
    long long item0 = 0;
    int phase0 = 0;
    for (int k = 0; k < n; ++k) {
        const ActiveCall &c = calls[k];
        soap_star *s = c.s;
        const int N = s->prm.grid_n, n_mu = s->prm.n_mu;
        const int ncap = ((N + 1) & ~1) + 2;
        const int job_cap = per_cell_cap(s, n_mu, ncap, n_kinds);
        int *d_njobs = s->d_sched.ptr, *d_work = d_njobs + c.n_phases;
        if (prepare) {
            RegionAtPhase *rp = reinterpret_cast<RegionAtPhase *>(h + rp_off) + rp_pos;
            localize_regions(s, c.regions, c.n_regions, c.phases, c.n_phases, c.radii, rp);
            PrepArgs a{};
            a.N = N;
            a.n_regions = c.n_regions;
            a.n_mu = n_mu;
            a.seg_cap = ncap;
            a.job_cap = job_cap;
            a.n_phases = c.n_phases;
            a.n_kinds = n_kinds;
            a.lb_types = (lb_is_one(c.spot) ? 0 : 2) | (lb_is_one(c.fac) ? 0 : 4);
            a.chunk_cols = std::max(32, (N + kPrepCluster - 1) / kPrepCluster);  // columns a CTA of the cluster may own
            a.rp = reinterpret_cast<const RegionAtPhase *>(d + rp_off) + rp_pos;
            a.mu = s->d_mu.ptr;
            a.w = s->d_w.ptr;
            a.col_a = s->d_col_a.ptr;
            a.bin = s->d_bin.ptr;
            a.lb.c[1][0] = 1.0;
            a.lb.c[2][0] = 1.0;
            if (use_lb && c.spot) { a.lb.c[1][0] = c.spot->lb_c0; a.lb.c[1][1] = c.spot->lb_c1; a.lb.c[1][2] = c.spot->lb_c2; }
            if (use_lb && c.fac) { a.lb.c[2][0] = c.fac->lb_c0; a.lb.c[2][1] = c.fac->lb_c1; a.lb.c[2][2] = c.fac->lb_c2; }
            a.ent = s->d_aent.ptr;
            a.seg_count = s->d_segcnt.ptr;
            a.n_active = s->d_nactive.ptr;
            a.jobs = s->d_jobs.ptr;
            a.n_jobs = d_njobs;
            a.work = d_work;
            a.counters = s->d_counters.ptr;
            hp[k] = a;
            hph[k] = phase0;
            rp_pos += (size_t)c.n_regions * c.n_phases;
            phase0 += c.n_phases;
        }
        f32::StarBlock b{};
        b.base[0] = static_cast<const float *>(c.q->data);
        b.base[1] = (c.spot && !quiet_rows) ? static_cast<const float *>(c.spot->data) : b.base[0];
        b.base[2] = (c.fac && !quiet_rows) ? static_cast<const float *>(c.fac->data) : b.base[0];
        b.contrast[1] = (c.spot && use_contrast) ? static_cast<const float *>(c.spot->contrast) : nullptr;
        b.contrast[2] = (c.fac && use_contrast) ? static_cast<const float *>(c.fac->contrast) : nullptr;
        b.pitch = c.q->pitch;
        b.row_len = s->clip_override > 0 ? s->clip_override : c.q->pitch;
        b.out_lo = s->out_lo_override >= 0 ? s->out_lo_override : 0;
        b.out_hi = s->out_hi_override >= 0 ? s->out_hi_override : c.q->n_pix;
        b.n_pix = c.q->n_pix;
        b.c0 = c.q->lambda0 / c.q->dlambda;
        b.n_mu = n_mu;
        b.halo = halo_for(s, c.q);
        b.ent = reinterpret_cast<const float2 *>(s->d_aent.ptr);
        b.n_tiles = (int)((c.q->n_pix + f32::kTile - 1) / f32::kTile);
        b.jobs = s->d_jobs.ptr;
        b.n_jobs = d_njobs;
        b.work = d_work;
        b.job_cap = job_cap;
        b.n_phases = c.n_phases;
        b.out = static_cast<float *>(c.out);
        if (all_effects) {
            b.out_fc[0] = static_cast<float *>(c.out_flux);
            b.out_fc[1] = static_cast<float *>(c.out_cb);
        }
        b.out_pitch = c.out_pitch;
        b.item0 = item0;
        hb[k] = b;
        item0 += (long long)c.n_phases * b.n_tiles;
        s->last_tile_px = f32::kTile;
    }
    const f32::StarBlock first_block = hb[0];
    if (prepare && !inline_rp) {
        hph[n] = phase0;
        SOAP_CUDA(own, cudaMemcpyAsync(d, h, total, cudaMemcpyHostToDevice, st));
    } else if (n > 1) {
        SOAP_CUDA(own, cudaMemcpyAsync(d + blk_off, h + blk_off, (size_t)n * sizeof(f32::StarBlock), cudaMemcpyHostToDevice, st));
    }
    if (stage) {
        SOAP_CUDA(own, cudaEventRecord(slot.done, st));
        slot.in_flight = true;
    }

    if (prepare && total_phases > 0) {
        // a4: one cluster of CTAs per (star, phase) bins, compacts and schedules (active.cuh).  CTAs of 512 threads while
        // every cluster of the launch is resident at once, smaller ones beyond that (see the kernel's header).
        const int threads = total_phases * kPrepCluster <= 2LL * own->n_sm ? 512 : 256;
        const dim3 grid((unsigned)(total_phases * kPrepCluster));
        auto launch_map = [&](auto tag) -> int {
            constexpr int T = decltype(tag)::value;
            const int slot = (T == 512 ? 0 : 1) * 2 + (inline_rp ? 1 : 0);
            if (inline_rp) {
                if (!own->attr_prep_set[slot]) {
                    SOAP_CUDA(own, (cudaFuncSetAttribute(active_prepare_kernel<float2, kInlineRegions, T>,
                                                         cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)));
                    own->attr_prep_set[slot] = true;
                }
                InlineRegions<kInlineRegions> inl;
                std::memcpy(inl.r, h + rp_off, n_rp * sizeof(RegionAtPhase));
                SOAP_CUDA(own, launch_pdl(active_prepare_kernel<float2, kInlineRegions, T>, grid, dim3(T), prep_smem, st, hp[0],
                                          (const PrepArgs *)nullptr, (const int *)nullptr, 1, inl));
            } else {
                if (!own->attr_prep_set[slot]) {
                    SOAP_CUDA(own, (cudaFuncSetAttribute(active_prepare_kernel<float2, 0, T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                         200 * 1024)));
                    own->attr_prep_set[slot] = true;
                }
                PrepArgs none{};
                InlineRegions<0> no_inl{};
                SOAP_CUDA(own, launch_pdl(active_prepare_kernel<float2, 0, T>, grid, dim3(T), prep_smem, st, none,
                                          reinterpret_cast<const PrepArgs *>(d + prep_off), reinterpret_cast<const int *>(d + ph_off), n,
                                          no_inl));
            }
            return SOAP_OK;
        };
        int rcm;
        if (threads == 512) rcm = launch_map(std::integral_constant<int, 512>{});
        else rcm = launch_map(std::integral_constant<int, 256>{});
        if (rcm) return rcm;
        SOAP_LAUNCH_CHECK(own, "active_prepare_kernel");
    }
    if (n_items == 0 || map_only) return SOAP_OK;
    // a5 + a6: persistent CTAs over the (star, phase, tile) items
    f32::Params p{};
    p.one = first_block;
    p.many = n > 1 ? reinterpret_cast<const f32::StarBlock *>(d + blk_off) : nullptr;
    p.n_stars = n;
    p.n_items = n_items;
    p.halo = max_halo;
    f32::set_layout(p);
    p.collapse = own->form_used == SOAP_FORM_FIR ? 1 : 0;
    p.item_counters = reinterpret_cast<int *>(&own->d_counters.ptr->item_next);
    if (all_effects) {
        using f32::eff_code;
        using f32::sia_f32_kernel;
        using f32::kMulZero; using f32::kMulOne; using f32::kMulC; using f32::kMulOneMinusC;
        // the multipliers of every kind's partial sum P (sia_f32.cuh, Params::eff); quiet-row kinds carry the weight -w
        if (n_kinds == 4) {  // LB = 1: total = sum C A_t - Q, flux = sum (C - 1) Q_t, CB = sum A_t - Q
            p.eff[0] = eff_code(0, 1, kMulOne, kMulOneMinusC, kMulOne);
            p.eff[1] = eff_code(1, 1, kMulC, kMulZero, kMulOne);
            p.eff[2] = eff_code(2, 2, kMulC, kMulZero, kMulOne);
            p.eff[3] = eff_code(0, 2, kMulOne, kMulOneMinusC, kMulOne);
        } else {
            // a type with a limb-brightening law: its quiet rows weighted w LB (kinds 4, 5) serve flux only, its own rows
            // weighted w (kinds 6, 7) CB only; a type without one keeps the two-kind form above (its kinds 4-7 stay empty)
            const soap_spectra *tab[3] = {nullptr, calls[0].spot, calls[0].fac};
            for (int t = 1; t <= 2; ++t) {
                const int kq = t == 1 ? 0 : 3;
                if (lb_is_one(tab[t])) {
                    p.eff[kq] = eff_code(0, t, kMulOne, kMulOneMinusC, kMulOne);
                    p.eff[t] = eff_code(t, t, kMulC, kMulZero, kMulOne);
                } else {
                    p.eff[kq] = eff_code(0, 0, kMulOne, kMulOne, kMulOne);
                    p.eff[t] = eff_code(t, t, kMulC, kMulZero, kMulZero);
                }
                p.eff[3 + t] = eff_code(0, t, kMulZero, kMulC, kMulZero);
                p.eff[5 + t] = eff_code(t, 0, kMulZero, kMulZero, kMulOne);
            }
        }
        if (!own->attr_effects_set) {
            SOAP_CUDA(own, (cudaFuncSetAttribute(sia_f32_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024)));
            own->attr_effects_set = true;
        }
        if (own->occ_effects_smem != smem) {
            int occ = 0;
            SOAP_CUDA(own, (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sia_f32_kernel<true, true>, f32::kThreads, smem)));
            if (occ < 1) return own->fail(SOAP_ERR_UNSUPPORTED, "active kernel does not fit on an SM (halo %d)", max_halo);
            own->occ_effects = occ;
            own->occ_effects_smem = smem;
        }
        const long long G = std::max(1LL, std::min((long long)own->n_sm * own->occ_effects, n_items));
        p.item_chunk = 1;
        p.order_phases = n_items > 2 * G ? 1 : 0;
        if (own->opt_timing) {
            for (int k = 2; k < 4; ++k)
                if (!own->ev[k]) SOAP_CUDA(own, cudaEventCreate(&own->ev[k]));
            SOAP_CUDA(own, cudaEventRecord(own->ev[2], st));
        }
        SOAP_CUDA(own, launch_pdl(sia_f32_kernel<true, true>, dim3((unsigned)G), dim3(f32::kThreads), smem, st, p));
        SOAP_LAUNCH_CHECK(own, "sia_f32_kernel<effects>");
        if (own->opt_timing) {
            SOAP_CUDA(own, cudaEventRecord(own->ev[3], st));
            own->ev_valid[1] = true;
        }
        return SOAP_OK;
    }
    if (!own->attr_active_set) {
        SOAP_CUDA(own, cudaFuncSetAttribute(f32::sia_f32_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        own->attr_active_set = true;
    }
    if (own->occ_active_smem != smem) {  // the occupancy query is cached per shared-memory size
        int occ = 0;
        SOAP_CUDA(own, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f32::sia_f32_kernel<true>, f32::kThreads, smem));
        if (occ < 1) return own->fail(SOAP_ERR_UNSUPPORTED, "active kernel does not fit on an SM (halo %d)", max_halo);
        own->occ_active = occ;
        own->occ_active_smem = smem;
    }
    const long long G = std::max(1LL, std::min((long long)own->n_sm * own->occ_active, n_items));
    // very long item lists (a batch of stars) are handed out several items at a time
    p.item_chunk = (int)std::max(1LL, std::min((long long)f32::kMaxItemChunk, n_items / (G * 64)));
    p.order_phases = n_items > 2 * G ? 1 : 0;  // with an item or two per CTA the order of the hand-out buys nothing
    if (own->opt_timing) {
        for (int k = 2; k < 4; ++k)
            if (!own->ev[k]) SOAP_CUDA(own, cudaEventCreate(&own->ev[k]));
        SOAP_CUDA(own, cudaEventRecord(own->ev[2], st));
    }
    SOAP_CUDA(own, launch_pdl(f32::sia_f32_kernel<true>, dim3((unsigned)G), dim3(f32::kThreads), smem, st, p));
    SOAP_LAUNCH_CHECK(own, "sia_f32_kernel<active>");
    if (own->opt_timing) {
        SOAP_CUDA(own, cudaEventRecord(own->ev[3], st));
        own->ev_valid[1] = true;
    }
    return SOAP_OK;
}

template <typename T>
int active_impl(soap_star *s, const soap_spectra *q, const soap_spectra *spot, const soap_spectra *fac,
                int n_regions, int n_phases, int effect, bool prepare, void *out, long long out_pitch, cudaStream_t st) {
    // (fp64 I/O, and fp32 under differential rotation; fp32 with solid-body rotation goes through active_f32_launch)
    // The three effects of Eq. 1-3 differ only in which table, weight and contrast an active entry uses:
    //   total: S_t, w LB_t(mu), C_t;   flux only: S_quiet, w LB_t(mu), C_t;   CB only: S_t, w, 1.
    // `prepare` = false reuses the entry lists of the previous pass (same weights).
    const bool use_lb = effect != SOAP_EFFECT_CB, use_contrast = effect != SOAP_EFFECT_CB;
    const bool quiet_rows = effect == SOAP_EFFECT_FLUX;
    using Ent = typename SiaTraits<T>::Ent;
    constexpr int TP = sia_tile_px<T>();
    const int N = s->prm.grid_n, n_mu = s->prm.n_mu;
    const int ncap = ((N + 1) & ~1) + 2;
    const long long n_seg = (long long)n_phases * 3 * n_mu;
    if (n_seg * ncap >= (1LL << 31)) return s->fail(SOAP_ERR_UNSUPPORTED, "n_phases * 3 * n_mu * N too large for one call");
    SOAP_CUDA(s, s->d_aent.reserve((size_t)n_seg * ncap * sizeof(Ent) + 64));
    SOAP_CUDA(s, s->d_segcnt.reserve((size_t)n_seg));
    SOAP_CUDA(s, s->d_nactive.reserve((size_t)n_phases));
    if (!s->d_counters.ptr) {
        SOAP_CUDA(s, s->d_counters.reserve(1));
        SOAP_CUDA(s, cudaMemsetAsync(s->d_counters.ptr, 0, sizeof(ActiveCounters), st));  // once per handle
    }
    const int job_cap = per_cell_cap(s, n_mu, ncap);
    SOAP_CUDA(s, s->d_jobs.reserve((size_t)n_phases * job_cap));
    SOAP_CUDA(s, s->d_sched.reserve((size_t)2 * n_phases));
    int *d_njobs = s->d_sched.ptr, *d_work = d_njobs + n_phases;
    s->last_n_phases = n_phases;
    const bool per_cell = s->prm.diff_rot != 0.0;  // the cells of a column no longer share a velocity (R-DR)
    // fp64 I/O under differential rotation: the generic kernel reads fixed slots of seg_cap entries per segment, so every
    // segment gets room for all the covered cells of a phase (fp64 is the small-configuration path)
    const long long cell_seg_cap = (per_cell && sizeof(T) != 4) ? ((s->active_pool_cap / 2 + 2) & ~1LL) : 0;
    if (per_cell && prepare) {
        const long long pool = cell_seg_cap > 0 ? cell_seg_cap * 3 * n_mu : s->active_pool_cap;
        if ((long long)n_phases * pool >= (1LL << 31)) return s->fail(SOAP_ERR_UNSUPPORTED, "n_phases * entries per phase too large for one call");
        SOAP_CUDA(s, s->d_aent.reserve((size_t)n_phases * pool * sizeof(Ent) + 64));
        PrepArgs a{};
        a.N = N;
        a.n_regions = n_regions;
        a.n_mu = n_mu;
        a.n_kinds = 3;
        a.seg_cap = (int)cell_seg_cap;
        a.n_phases = n_phases;
        a.pool_cap = (int)pool;
        a.job_cap = 3 * n_mu + (int)(pool / kActiveJobCap) + 2;
        SOAP_CUDA(s, s->d_jobs.reserve((size_t)n_phases * a.job_cap));
        a.chunk_cols = std::max(32, (N + kPrepCluster - 1) / kPrepCluster);
        if (prep_cells_smem_bytes(n_mu, a.chunk_cols) > 200 * 1024)
            return s->fail(SOAP_ERR_UNSUPPORTED, "grid_n %d with %d mu bins exceeds the active-map kernel's shared memory", N, n_mu);
        a.rp = s->d_rp.ptr;
        a.mu = s->d_mu.ptr;
        a.w = s->d_w.ptr;
        a.col_a = s->d_col_a.ptr;
        a.bin = s->d_bin.ptr;
        a.vel = s->d_vel.ptr;
        a.mode = s->prm.doppler_mode;
        a.lb.c[1][0] = 1.0;
        a.lb.c[2][0] = 1.0;
        if (use_lb && spot) { a.lb.c[1][0] = spot->lb_c0; a.lb.c[1][1] = spot->lb_c1; a.lb.c[1][2] = spot->lb_c2; }
        if (use_lb && fac) { a.lb.c[2][0] = fac->lb_c0; a.lb.c[2][1] = fac->lb_c1; a.lb.c[2][2] = fac->lb_c2; }
        a.ent = s->d_aent.ptr;
        a.seg_count = cell_seg_cap > 0 ? s->d_segcnt.ptr : nullptr;
        a.n_active = s->d_nactive.ptr;
        a.jobs = s->d_jobs.ptr;
        a.n_jobs = d_njobs;
        a.work = d_work;
        a.counters = s->d_counters.ptr;
        const size_t smem = prep_cells_smem_bytes(n_mu, a.chunk_cols);
        SOAP_CUDA(s, cudaFuncSetAttribute(active_prepare_cells_kernel<Ent>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        active_prepare_cells_kernel<Ent><<<n_phases * kPrepCluster, kPrepThreads, smem, st>>>(a);
        SOAP_LAUNCH_CHECK(s, "active_prepare_cells_kernel");
    } else if (prepare) {
        // a4 in one launch: one cluster of CTAs per phase bins, compacts and schedules (active.cuh)
        PrepArgs a{};
        a.N = N;
        a.n_regions = n_regions;
        a.n_mu = n_mu;
        a.n_kinds = 3;
        a.seg_cap = ncap;
        a.job_cap = job_cap;
        a.n_phases = n_phases;
        a.chunk_cols = std::max(32, (N + kPrepCluster - 1) / kPrepCluster);  // columns a CTA of the cluster may own
        if (prep_smem_bytes(n_mu, a.chunk_cols, N, n_regions) > 200 * 1024)
            return s->fail(SOAP_ERR_UNSUPPORTED, "grid_n %d with %d mu bins exceeds the active-map kernel's shared memory", N, n_mu);
        a.rp = s->d_rp.ptr;
        a.mu = s->d_mu.ptr;
        a.w = s->d_w.ptr;
        a.col_a = s->d_col_a.ptr;
        a.bin = s->d_bin.ptr;
        a.lb.c[1][0] = 1.0;
        a.lb.c[2][0] = 1.0;
        if (use_lb && spot) { a.lb.c[1][0] = spot->lb_c0; a.lb.c[1][1] = spot->lb_c1; a.lb.c[1][2] = spot->lb_c2; }
        if (use_lb && fac) { a.lb.c[2][0] = fac->lb_c0; a.lb.c[2][1] = fac->lb_c1; a.lb.c[2][2] = fac->lb_c2; }
        a.ent = s->d_aent.ptr;
        a.seg_count = s->d_segcnt.ptr;
        a.n_active = s->d_nactive.ptr;
        a.jobs = s->d_jobs.ptr;
        a.n_jobs = d_njobs;
        a.work = d_work;
        a.counters = s->d_counters.ptr;
        const size_t smem = prep_smem_bytes(n_mu, a.chunk_cols, N, n_regions);
        SOAP_CUDA(s, (cudaFuncSetAttribute(active_prepare_kernel<Ent, 0, kPrepThreads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)));
        InlineRegions<0> no_inl{};
        active_prepare_kernel<Ent, 0, kPrepThreads><<<n_phases * kPrepCluster, kPrepThreads, smem, st>>>(a, nullptr, nullptr, 1, no_inl);
        SOAP_LAUNCH_CHECK(s, "active_prepare_kernel");
    }
    if (sizeof(T) == 4) {
        ActiveCall c{s, q, spot, fac, nullptr, n_regions, nullptr, n_phases, nullptr, out, out_pitch};
        return active_f32_launch(&c, 1, effect, false, true, st);
    }
    SiaParams<T> p{};
    p.base[0] = static_cast<const T *>(q->data);
    p.base[1] = (spot && !quiet_rows) ? static_cast<const T *>(spot->data) : p.base[0];
    p.base[2] = (fac && !quiet_rows) ? static_cast<const T *>(fac->data) : p.base[0];
    p.contrast[1] = (spot && use_contrast) ? static_cast<const T *>(spot->contrast) : nullptr;
    p.contrast[2] = (fac && use_contrast) ? static_cast<const T *>(fac->contrast) : nullptr;
    p.pitch = q->pitch;
    p.n_pix = q->n_pix;
    p.c0 = q->lambda0 / q->dlambda;
    p.n_mu = n_mu;
    p.halo = halo_for(s, q);
    p.ent = reinterpret_cast<const Ent *>(s->d_aent.ptr);
    p.seg_count = s->d_segcnt.ptr;
    p.seg_cap = per_cell ? (int)cell_seg_cap : ncap;
    p.out = static_cast<T *>(out);
    p.out_pitch = out_pitch;
    const int n_tiles = (int)((q->n_pix + TP - 1) / TP);
    s->last_tile_px = TP;
    return launch_sia<T, true>(s, p, dim3(n_tiles, n_phases), st);
}

int check_regions(soap_star *s, const soap_region *regions, int n_regions, const double *phases, int n_phases,
                  const soap_spectra *spot, const soap_spectra *fac) {
    if (n_regions < 0 || n_phases < 0) return s->fail(SOAP_ERR_INVALID_ARG, "negative n_regions / n_phases");
    if (n_regions > 0 && !regions) return s->fail(SOAP_ERR_INVALID_ARG, "regions is NULL");
    if (n_phases > 0 && !phases) return s->fail(SOAP_ERR_INVALID_ARG, "phases is NULL");
    for (int r = 0; r < n_regions; ++r) {
        const soap_region &g = regions[r];
        if (g.type != SOAP_SPOT && g.type != SOAP_FACULA) return s->fail(SOAP_ERR_INVALID_ARG, "region %d: unknown type %d", r, g.type);
        if (!(g.radius > 0.0 && g.radius < 1.0)) return s->fail(SOAP_ERR_INVALID_ARG, "region %d: radius must be in (0,1)", r);
        if (!std::isfinite(g.lat_deg) || !std::isfinite(g.lon_deg)) return s->fail(SOAP_ERR_INVALID_ARG, "region %d: lat/lon not finite", r);
        if (g.type == SOAP_SPOT && !spot) return s->fail(SOAP_ERR_INVALID_ARG, "region %d is a spot but spot spectra are NULL", r);
        if (g.type == SOAP_FACULA && !fac) return s->fail(SOAP_ERR_INVALID_ARG, "region %d is a facula but facula spectra are NULL", r);
    }
    for (int p = 0; p < n_phases; ++p)
        if (!std::isfinite(phases[p])) return s->fail(SOAP_ERR_INVALID_ARG, "phase %d not finite", p);
    return SOAP_OK;
}

// upload_region_centres: the same for the calls that are not batched (fp64 I/O, differential rotation).
// `radii` (nullable): HOST [n_phases][n_regions] radius of every region at every phase (evolving regions);
// <= 0 means the region is absent at that phase.  NULL: regions[r].radius at every phase.
int upload_region_centres(soap_star *s, const soap_region *regions, int n_regions, const double *phases,
                          int n_phases, const double *radii, cudaStream_t st) {
    {
        // per-cell form: a region's covered cells lie in a disc of radius chord = 2 sin(alpha / 2) around its projected
        // centre; with the cell-centre rule at most pi (chord N / 2 + 1.5)^2 of them, two entries each
        const double pi_ = 3.14159265358979323846, half = 0.5 * (double)s->prm.grid_n;
        double cells = 0.0;
        for (int r = 0; r < n_regions; ++r) {
            double rad = regions[r].radius;
            if (radii) {
                rad = 0.0;
                for (int p = 0; p < n_phases; ++p) rad = std::max(rad, radii[(size_t)p * n_regions + r]);
            }
            const double ch = 2.0 * std::sin(0.5 * std::asin(rad)) * half + 1.5;
            cells += pi_ * ch * ch;
        }
        cells = std::min(cells, (double)s->prm.grid_n * (double)s->prm.grid_n);
        s->active_pool_cap = ((2LL * (long long)std::ceil(cells) + 2LL * 3 * s->prm.n_mu + 8) + 1) & ~1LL;
    }
    const size_t n = (size_t)n_regions * n_phases;
    if (n == 0) return SOAP_OK;
    soap_star::PinnedSlot &slot = s->h_rp[s->h_rp_next];
    s->h_rp_next = (s->h_rp_next + 1) & 3;
    if (slot.in_flight) {
        SOAP_CUDA(s, cudaEventSynchronize(slot.done));
        slot.in_flight = false;
    }
    if (!slot.done) SOAP_CUDA(s, cudaEventCreateWithFlags(&slot.done, cudaEventDisableTiming));
    if (n > slot.cap) {
        if (slot.ptr) cudaFreeHost(slot.ptr);
        slot.ptr = nullptr;
        slot.cap = 0;
        SOAP_CUDA(s, cudaMallocHost(reinterpret_cast<void **>(&slot.ptr), n * sizeof(RegionAtPhase)));
        slot.cap = n;
    }
    if (n > s->d_rp.cap) {
        // growing d_rp frees the old buffer, which an earlier call's kernel may still be reading
        SOAP_CUDA(s, cudaDeviceSynchronize());
        SOAP_CUDA(s, s->d_rp.reserve(n));
    }
    localize_regions(s, regions, n_regions, phases, n_phases, radii, slot.ptr);
    SOAP_CUDA(s, cudaMemcpyAsync(s->d_rp.ptr, slot.ptr, n * sizeof(RegionAtPhase), cudaMemcpyHostToDevice, st));
    SOAP_CUDA(s, cudaEventRecord(slot.done, st));
    slot.in_flight = true;
    return SOAP_OK;
}


// soap_synthesize_host for long fp32 spectra: the wavelength axis is cut into chunks of whole tiles, and the upload of
// chunk c+1, the kernels of chunk c and the download of chunk c-1 overlap on three streams (every output pixel depends
// only on source pixels within the halo, so a chunk is the same computation on a window [m0 - Hc, m1 + Hc) of the
// tables; only its interior [m0, m1) is kept).  The PCIe copies, not the kernels, bound this entry point.
int synthesize_host_pipelined(soap_star *s, const soap_star_params *prm, const soap_spectra *quiet, const soap_spectra *spot,
                              const soap_spectra *facula, const soap_region *regions, int32_t n_regions, const double *phases,
                              int32_t n_phases, void *out_quiet, void *out_delta, int32_t *n_active, cudaStream_t st) {
    const soap_spectra *in[3] = {quiet, spot, facula};
    const long long P = quiet->n_pix, pitch = quiet->pitch;
    for (int k = 1; k < 3; ++k) {
        if (!in[k]) continue;
        if (!in[k]->data || in[k]->n_pix != P || in[k]->pitch != pitch || in[k]->dtype != SOAP_F32)
            return s->fail(SOAP_ERR_INVALID_ARG, "spectra %d: data / n_pix / pitch / dtype differ from quiet", k);
    }
    // every argument is checked before anything is enqueued (the tables are HOST memory here: the device-side alignment
    // rule applies to the staged copies, which the library aligns itself)
    for (int k = 0; k < 3; ++k) {
        if (!in[k]) continue;
        soap_spectra probe = *in[k];
        probe.data = reinterpret_cast<const void *>(static_cast<uintptr_t>(256));
        int rcv = check_spectra(s, &probe, k == 0 ? "quiet" : k == 1 ? "spot" : "facula");
        if (rcv) return rcv;
        if (k > 0 && (in[k]->lambda0 != quiet->lambda0 || in[k]->dlambda != quiet->dlambda))
            return s->fail(SOAP_ERR_INVALID_ARG, "spectra %d: lambda0 / dlambda differ from quiet", k);
    }
    int rc = soap_disk_geometry(s, prm, st, nullptr);
    if (rc) return rc;
    // the (small) region upload goes first: copies of one direction are served in issue order, and behind the table
    // uploads it would hold back the first chunk's kernels until every table has arrived
    if ((rc = check_regions(s, regions, n_regions, phases, n_phases, spot, facula))) return rc;
    const bool map_first = prm->diff_rot == 0.0;  // solid body: the active map is built here, ahead of the table uploads
    if (map_first) {
        ActiveCall c{s, quiet, spot, facula, regions, n_regions, phases, n_phases, nullptr, nullptr, P};
        if ((rc = active_f32_launch(&c, 1, SOAP_EFFECT_TOTAL, true, false, st, true))) return rc;
    } else if ((rc = upload_region_centres(s, regions, n_regions, phases, n_phases, nullptr, st))) {
        return rc;
    }
    if (!s->s_h2d) SOAP_CUDA(s, cudaStreamCreateWithFlags(&s->s_h2d, cudaStreamNonBlocking));
    if (!s->s_d2h) SOAP_CUDA(s, cudaStreamCreateWithFlags(&s->s_d2h, cudaStreamNonBlocking));
    const long long tiles = (P + f32::kTile - 1) / f32::kTile;
    const int K = (int)std::max(1LL, std::min(4LL, tiles / 32));  // measured: 3-4 chunks are best, more only add copies
    const long long Lc = ((tiles + K - 1) / K) * f32::kTile;  // chunk length: whole tiles
    const long long Hc = halo_for(s, quiet) + 4;              // halo of the whole spectrum (a multiple of 4)
    while ((int)s->ev_pipe.size() < 1 + 3 * K) {
        cudaEvent_t e;
        SOAP_CUDA(s, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        s->ev_pipe.push_back(e);
    }
    cudaEvent_t ev_start = s->ev_pipe[0];
    auto ev_up = [&](int c) { return s->ev_pipe[1 + c]; };
    auto ev_done = [&](int c) { return s->ev_pipe[1 + K + c]; };
    auto ev_out = [&](int c) { return s->ev_pipe[1 + 2 * K + c]; };
    for (int k = 0; k < 3; ++k) {
        if (!in[k]) continue;
        SOAP_CUDA(s, s->d_stage[k].reserve((size_t)prm->n_mu * pitch * 4));
        if (k > 0 && in[k]->contrast) SOAP_CUDA(s, s->d_stage_c[k].reserve((size_t)P * 4));
    }
    // Results go straight to the caller's arrays when those are pinned (device-visible) host memory: the kernels' stores
    // cross PCIe while the next chunk's tables come in, and no device-to-host copy is queued at all.  Pageable outputs are
    // staged in device memory and copied back chunk by chunk.
    float *dq = nullptr, *dd = nullptr;
    {
        cudaPointerAttributes aq{}, ad{};
        const bool okq = cudaPointerGetAttributes(&aq, out_quiet) == cudaSuccess && aq.type == cudaMemoryTypeHost && aq.devicePointer;
        const bool okd = cudaPointerGetAttributes(&ad, out_delta) == cudaSuccess && ad.type == cudaMemoryTypeHost && ad.devicePointer;
        cudaGetLastError();  // a pageable pointer is reported as an error by older runtimes: not ours to keep
        if (okq && okd) {
            dq = static_cast<float *>(aq.devicePointer);
            dd = static_cast<float *>(ad.devicePointer);
        }
    }
    const bool zero_copy = dq != nullptr;
    if (!zero_copy) {
        SOAP_CUDA(s, s->d_out_q.reserve((size_t)P * 4));
        SOAP_CUDA(s, s->d_out_d.reserve((size_t)n_phases * P * 4));
        dq = reinterpret_cast<float *>(s->d_out_q.ptr);
        dd = reinterpret_cast<float *>(s->d_out_d.ptr);
    }
    // the copy streams start after whatever the caller's stream holds so far (buffers of an earlier call may be in use)
    SOAP_CUDA(s, cudaEventRecord(ev_start, st));
    SOAP_CUDA(s, cudaStreamWaitEvent(s->s_h2d, ev_start, 0));
    SOAP_CUDA(s, cudaStreamWaitEvent(s->s_d2h, ev_start, 0));
    // uploads: a partition of the columns, chunk c carrying [m0 + Hc, m1 + Hc) (the first from 0, the last up to P)
    for (int c = 0; c < K; ++c) {
        const long long m0 = c * Lc, m1 = std::min(P, m0 + Lc);
        const long long u0 = c == 0 ? 0 : std::min(P, m0 + Hc), u1 = c == K - 1 ? P : std::min(P, m1 + Hc);
        if (u1 > u0) {
            for (int k = 0; k < 3; ++k) {
                if (!in[k]) continue;
                SOAP_CUDA(s, cudaMemcpy2DAsync(reinterpret_cast<float *>(s->d_stage[k].ptr) + u0, (size_t)pitch * 4,
                                               static_cast<const float *>(in[k]->data) + u0, (size_t)pitch * 4, (size_t)(u1 - u0) * 4,
                                               (size_t)prm->n_mu, cudaMemcpyHostToDevice, s->s_h2d));
                if (k > 0 && in[k]->contrast)
                    SOAP_CUDA(s, cudaMemcpyAsync(reinterpret_cast<float *>(s->d_stage_c[k].ptr) + u0,
                                                 static_cast<const float *>(in[k]->contrast) + u0, (size_t)(u1 - u0) * 4,
                                                 cudaMemcpyHostToDevice, s->s_h2d));
            }
        }
        SOAP_CUDA(s, cudaEventRecord(ev_up(c), s->s_h2d));
    }
    for (int c = 0; c < K; ++c) {
        const long long m0 = c * Lc, m1 = std::min(P, m0 + Lc);
        if (m1 <= m0) {
            SOAP_CUDA(s, cudaEventRecord(ev_out(c), s->s_d2h));
            continue;
        }
        const long long v0 = std::max(0LL, m0 - Hc), v1 = std::min(P, m1 + Hc);  // the window this chunk computes on
        soap_spectra dev[3];
        for (int k = 0; k < 3; ++k) {
            if (!in[k]) continue;
            dev[k] = *in[k];
            dev[k].data = reinterpret_cast<float *>(s->d_stage[k].ptr) + v0;
            dev[k].n_pix = v1 - v0;
            dev[k].lambda0 = in[k]->lambda0 + (double)v0 * in[k]->dlambda;
            dev[k].contrast = (k > 0 && in[k]->contrast) ? reinterpret_cast<float *>(s->d_stage_c[k].ptr) + v0 : nullptr;
        }
        SOAP_CUDA(s, cudaStreamWaitEvent(st, ev_up(c), 0));
        s->clip_override = pitch - v0;
        s->out_lo_override = m0 - v0;  // the window's margins belong to the neighbouring chunks
        s->out_hi_override = m1 - v0;
        rc = soap_integrate_quiet(s, &dev[0], dq + v0, st);
        if (!rc) {
            s->reuse_lists = map_first || c > 0;  // the active map does not depend on the wavelength window
            s->regions_uploaded = true;
            rc = soap_active_timeseries(s, &dev[0], spot ? &dev[1] : nullptr, facula ? &dev[2] : nullptr, regions, n_regions, phases,
                                        n_phases, dd + v0, P, nullptr, st);
        }
        s->clip_override = 0;
        s->out_lo_override = s->out_hi_override = -1;
        s->reuse_lists = false;
        s->regions_uploaded = false;
        if (rc) {  // nothing of this call may still be in flight when the caller gets its buffers back
            cudaStreamSynchronize(st);
            cudaStreamSynchronize(s->s_h2d);
            cudaStreamSynchronize(s->s_d2h);
            return rc;
        }
        SOAP_CUDA(s, cudaEventRecord(ev_done(c), st));
        if (!zero_copy) {
            SOAP_CUDA(s, cudaStreamWaitEvent(s->s_d2h, ev_done(c), 0));
            SOAP_CUDA(s, cudaMemcpyAsync(static_cast<float *>(out_quiet) + m0, dq + m0, (size_t)(m1 - m0) * 4, cudaMemcpyDeviceToHost, s->s_d2h));
            SOAP_CUDA(s, cudaMemcpy2DAsync(static_cast<float *>(out_delta) + m0, (size_t)P * 4, dd + m0, (size_t)P * 4,
                                           (size_t)(m1 - m0) * 4, (size_t)n_phases, cudaMemcpyDeviceToHost, s->s_d2h));
        }
        SOAP_CUDA(s, cudaEventRecord(ev_out(c), s->s_d2h));
    }
    if (!zero_copy)
        for (int c = 0; c < K; ++c) SOAP_CUDA(s, cudaStreamWaitEvent(st, ev_out(c), 0));
    if (n_active) SOAP_CUDA(s, cudaMemcpyAsync(n_active, s->d_nactive.ptr, (size_t)n_phases * sizeof(int), cudaMemcpyDeviceToHost, st));
    SOAP_CUDA(s, cudaStreamSynchronize(st));
    return SOAP_OK;
}
}  // namespace

// ---- soap_integrate_quiet_static: the quiet spectrum without any device allocation ---------------------------------
// soap_integrate_quiet keeps its per-chunk fp64 partial sums in a buffer it (re)allocates with cudaMalloc when a call
// needs more than any call before it.  Some callers cannot afford that: a host application that has handed all of the
// device's memory to its own pool (cudaMalloc then simply fails), or a loop that must never stall (cudaMalloc and
// cudaFree synchronise the whole device).  For them the same two kernels (sia.cuh: sia_kernel<T, false>, reduce_partials_kernel<T>) run with their
// partial sums in the array below instead: fixed size, part of the library image, so every device that loads the library
// gives up these 4 MiB until the process exits, whether the entry point is ever called or not.
//
// Only device code may name the array directly.  In host code `g_static_partial` is a host-side shadow symbol, not a device
// address: the kernels are given what cudaGetSymbolAddress returns for the device that is current, looked up once per
// device (static_partial_address).
constexpr long long kStaticPartialDoubles = 512LL * 1024;  // 4 MiB of fp64 partial sums: n_splits * round_up4(n_pix) <= this
static __device__ __align__(256) double g_static_partial[kStaticPartialDoubles];

namespace {
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
double *g_static_partial_dev[kStaticMaxDevices] = {};  // device address of g_static_partial on device d (nullptr: not looked up)

// Device address of the static scratch on s->device.  The device must be current.  The first call on a device performs
// the look-up (which loads the library's module on that device if nothing has yet); later calls read the cached pointer.
int static_partial_address(soap_star *s, double **out) {
    if (s->device < 0 || s->device >= kStaticMaxDevices)
        return s->fail(SOAP_ERR_UNSUPPORTED, "static scratch: device %d is outside 0..%d", s->device, kStaticMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    double *&slot = g_static_partial_dev[s->device];
    if (!slot) {
        double *p = nullptr;
        SOAP_CUDA(s, cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_static_partial));
        if (!p) return s->fail(SOAP_ERR_CUDA, "cudaGetSymbolAddress returned a null address for the static scratch");
        slot = p;
    }
    *out = slot;
    return SOAP_OK;
}

template <typename T>
int quiet_static_impl(soap_star *s, const soap_spectra *q, void *out, cudaStream_t st) {
    constexpr int TP = sia_tile_px<T>();
    const long long P = q->n_pix;
    const long long part_pitch = (P + 3) & ~3LL;
    if (part_pitch > kStaticPartialDoubles)
        return s->fail(SOAP_ERR_UNSUPPORTED, "soap_integrate_quiet_static: n_pix = %lld exceeds the static scratch (at most %lld pixels); "
                       "use soap_integrate_quiet", P, kStaticPartialDoubles);
    const size_t smem = sia_smem_bytes<T>(halo_for(s, q));
    if (smem > 227 * 1024)
        return s->fail(SOAP_ERR_UNSUPPORTED, "shift of %d pixels needs %zu B of shared memory", halo_for(s, q), smem);
    double *partial = nullptr;
    int rc = static_partial_address(s, &partial);
    if (rc) return rc;
    const int n_tiles = (int)((P + TP - 1) / TP);
    // the entry list is cut into as many chunks as soap_integrate_quiet's generic path would take, capped by what the
    // static array holds
    int splits = s->opt_quiet_splits;
    if (splits <= 0) {
        splits = (int)std::lround((double)(s->n_sm * 8) / n_tiles);
        const long long max_entries = (long long)s->prm.grid_n * (s->cell_entries ? s->prm.grid_n : s->prm.n_mu);
        const int cap = (int)std::max(1LL, max_entries / 16);
        splits = std::max(1, std::min(std::min(splits, 256), cap));
    }
    splits = (int)std::max(1LL, std::min<long long>(splits, kStaticPartialDoubles / part_pitch));
    SiaParams<T> p{};
    p.base[0] = static_cast<const T *>(q->data);
    p.pitch = q->pitch;
    p.n_pix = P;
    p.c0 = q->lambda0 / q->dlambda;
    p.n_mu = s->prm.n_mu;
    p.halo = halo_for(s, q);
    if (sizeof(T) == 4) p.ent = reinterpret_cast<const typename SiaTraits<T>::Ent *>(s->d_ent32.ptr);
    else p.ent = reinterpret_cast<const typename SiaTraits<T>::Ent *>(s->d_ent64.ptr);
    p.row_start = s->d_row_start.ptr;
    p.n_splits = splits;
    p.partial = partial;
    p.part_pitch = part_pitch;
    if (smem > 48 * 1024)
        SOAP_CUDA(s, cudaFuncSetAttribute(sia_kernel<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // every partial[split][m], m < n_pix, is stored by the first launch before the second reads it: nothing in the array
    // has to start at zero, and what an earlier call left there is never read
    sia_kernel<T, false><<<dim3(n_tiles, splits), kThreads, smem, st>>>(p);
    SOAP_LAUNCH_CHECK(s, "sia_kernel<quiet> (static scratch)");
    const int threads = 256;
    const long long quads = (P + 3) / 4;
    reduce_partials_kernel<T><<<(unsigned)((quads + threads - 1) / threads), threads, 0, st>>>(partial, part_pitch, splits, P,
                                                                                             static_cast<T *>(out));
    SOAP_LAUNCH_CHECK(s, "reduce_partials_kernel (static scratch)");
    return SOAP_OK;
}
}  // namespace

extern "C" {

int soap_version(void) { return SOAP_B200_VERSION; }

const char *soap_last_error(const soap_star *star) { return star ? star->err.c_str() : g_create_error.c_str(); }

int soap_create(soap_star **out, int device) {
    if (!out) {
        g_create_error = "soap_create: out is NULL";
        return SOAP_ERR_INVALID_ARG;
    }
    *out = nullptr;
    int n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess || n_dev == 0) {
        g_create_error = std::string("soap_create: no CUDA device (") + cudaGetErrorString(e) + "); this library has no CPU fallback";
        return SOAP_ERR_CUDA;
    }
    if (device < 0 || device >= n_dev) {
        g_create_error = "soap_create: device index out of range";
        return SOAP_ERR_INVALID_ARG;
    }
    soap_star *s = new (std::nothrow) soap_star();
    if (!s) {
        g_create_error = "soap_create: out of host memory";
        return SOAP_ERR_OOM;
    }
    s->device = device;
    cudaSetDevice(device);
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device) == cudaSuccess && n_sm > 0) s->n_sm = n_sm;
    *out = s;
    return SOAP_OK;
}

int soap_destroy(soap_star *s) {
    if (!s) return SOAP_OK;
    cudaSetDevice(s->device);
    s->d_cWp.release(); s->d_chdr.release(); s->d_cstars.release(); s->d_gargs.release();
    s->d_geom_done.release(); s->d_colcnt.release(); s->d_cellpos.release(); s->d_mu.release(); s->d_w.release(); s->d_vel.release(); s->d_col_a.release();
    s->d_Wbin.release(); s->d_col_sumw.release(); s->d_bin.release(); s->d_col_nvis.release(); s->d_row_start.release();
    s->d_ent32.release(); s->d_ent64.release(); s->d_info.release(); s->d_partial.release(); s->d_tile_ticket.release(); s->d_rp.release();
    s->d_aent.release(); s->d_segcnt.release(); s->d_nactive.release(); s->d_counters.release(); s->d_sched.release(); s->d_jobs.release();
    for (int k = 0; k < 3; ++k) { s->d_stage[k].release(); s->d_stage_c[k].release(); }
    s->d_out_q.release(); s->d_out_d.release();
    for (auto &e : s->ev)
        if (e) cudaEventDestroy(e);
    for (auto &e : s->ev_pipe) cudaEventDestroy(e);
    if (s->s_h2d) cudaStreamDestroy(s->s_h2d);
    if (s->s_d2h) cudaStreamDestroy(s->s_d2h);
    for (auto &slot : s->h_rp) {
        if (slot.ptr) cudaFreeHost(slot.ptr);
        if (slot.done) cudaEventDestroy(slot.done);
    }
    for (auto &slot : s->h_call) {
        if (slot.ptr) cudaFreeHost(slot.ptr);
        if (slot.done) cudaEventDestroy(slot.done);
    }
    s->d_call.release();
    delete s;
    return SOAP_OK;
}

int soap_set_option(soap_star *s, int32_t option, int64_t value) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    switch (option) {
        case SOAP_OPT_FORM:
            if (value < SOAP_FORM_AUTO || value > SOAP_FORM_COMPOSITE) return s->fail(SOAP_ERR_INVALID_ARG, "unknown form %lld", (long long)value);
            if ((int)value != s->form) s->ready = false;  // entry list must be rebuilt
            s->form = (int)value;
            return SOAP_OK;
        case SOAP_OPT_QUIET_SPLITS:
            if (value < 0 || value > 1024) return s->fail(SOAP_ERR_INVALID_ARG, "quiet splits out of range");
            s->opt_quiet_splits = (int)value;
            return SOAP_OK;
        case SOAP_OPT_KERNEL_TIMING:
            s->opt_timing = value != 0;
            s->ev_valid[0] = s->ev_valid[1] = false;
            return SOAP_OK;
        case SOAP_OPT_EFFECT_PASSES:
            s->opt_effect_passes = value != 0;
            return SOAP_OK;
        default:
            return s->fail(SOAP_ERR_INVALID_ARG, "unknown option %d", option);
    }
}

// soap_disk_geometry in three parts, so that the batch entry point can check every star before anything is enqueued and
// launch once for all of them: argument checks; state, scratch and the kernel's arguments; what follows the launch.
static int geometry_check(soap_star *s, const soap_star_params *prm) {
    if (!prm) return s->fail(SOAP_ERR_INVALID_ARG, "params is NULL");
    if (prm->grid_n < 1 || prm->grid_n > 8192) return s->fail(SOAP_ERR_INVALID_ARG, "grid_n must be in 1..8192");
    if (prm->n_mu < 1 || prm->n_mu > SOAP_MAX_MU) return s->fail(SOAP_ERR_INVALID_ARG, "n_mu must be in 1..%d", SOAP_MAX_MU);
    if (!prm->mu_centres) return s->fail(SOAP_ERR_INVALID_ARG, "mu_centres is NULL");
    for (int b = 0; b < prm->n_mu; ++b) {
        if (!std::isfinite(prm->mu_centres[b])) return s->fail(SOAP_ERR_INVALID_ARG, "mu_centres[%d] not finite", b);
        if (b && !(prm->mu_centres[b] > prm->mu_centres[b - 1])) return s->fail(SOAP_ERR_INVALID_ARG, "mu_centres must be strictly ascending");
    }
    if (!std::isfinite(prm->vsini_kms) || !std::isfinite(prm->incl_deg) || !std::isfinite(prm->ld_u1) || !std::isfinite(prm->ld_u2))
        return s->fail(SOAP_ERR_INVALID_ARG, "vsini / incl / limb-darkening coefficients must be finite");
    if (prm->doppler_mode != 0 && prm->doppler_mode != 1) return s->fail(SOAP_ERR_INVALID_ARG, "doppler_mode must be 0 or 1");
    const double pi = 3.14159265358979323846;
    const double sini = std::sin(prm->incl_deg * pi / 180.0), cosi = std::cos(prm->incl_deg * pi / 180.0);
    if (std::fabs(prm->vsini_kms * sini) * std::max(1.0, 1.0 + prm->diff_rot) >= 0.1 * kSpeedOfLightKms)
        return s->fail(SOAP_ERR_INVALID_ARG, "|v| must be below 0.1 c");

    if (!std::isfinite(prm->diff_rot) || !(prm->diff_rot > -1.0)) return s->fail(SOAP_ERR_INVALID_ARG, "diff_rot must be finite and > -1");
    if (prm->diff_rot != 0.0 && s->form == SOAP_FORM_BINNED)
        return s->fail(SOAP_ERR_UNSUPPORTED, "SOAP_FORM_BINNED needs solid-body rotation: the cells of a column must share one velocity");
    if (prm->diff_rot != 0.0 && s->form == SOAP_FORM_COMPOSITE)
        return s->fail(SOAP_ERR_UNSUPPORTED, "SOAP_FORM_COMPOSITE needs solid-body rotation: the cells of a column must share one velocity");
    return SOAP_OK;
}

static int geometry_prepare(soap_star *s, const soap_star_params *prm, cudaStream_t st, GeomArgs &ga, size_t &fin_bytes_out) {
    const double pi = 3.14159265358979323846;
    const double sini = std::sin(prm->incl_deg * pi / 180.0), cosi = std::cos(prm->incl_deg * pi / 180.0);
    SOAP_CUDA(s, cudaSetDevice(s->device));
    s->ready = false;
    s->last_form = 0;
    s->prm = *prm;
    s->mu_centres.assign(prm->mu_centres, prm->mu_centres + prm->n_mu);
    s->prm.mu_centres = s->mu_centres.data();
    s->sini = sini;
    s->cosi = cosi;
    const int N = prm->grid_n, n_mu = prm->n_mu;
    const size_t ncell = (size_t)N * N;
    s->form_used = (s->form == SOAP_FORM_CELLS || s->form == SOAP_FORM_FIR) ? s->form : SOAP_FORM_BINNED;
    // the composite-column form holds every mu-bin row of a span in registers: up to comp::kMaxBins bins
    // AUTO takes it for the quiet spectrum whenever it applies: its cost does not depend on v sin i, and it is at least as
    // fast as the binned entries at every v sin i measured (C3: 0.133 vs 0.140 ms at 2 km/s, 0.143 vs 0.297 ms at 20 km/s)
    if ((s->form == SOAP_FORM_COMPOSITE || s->form == SOAP_FORM_AUTO) && prm->diff_rot == 0.0 && n_mu_ok_for_composite(prm->n_mu))
        s->form_used = SOAP_FORM_COMPOSITE;
    s->cell_entries = s->form == SOAP_FORM_CELLS || prm->diff_rot != 0.0;
    // AUTO under differential rotation: per-cell entries with every run collapsed (the binned form does not apply;
    // the collapse is exact and ~5x cheaper than one lerp-accumulate per cell and pixel)
    if (s->cell_entries && s->form_used == SOAP_FORM_BINNED) s->form_used = s->form == SOAP_FORM_AUTO ? SOAP_FORM_FIR : SOAP_FORM_CELLS;
    const double vmax = std::fabs(prm->vsini_kms * sini) * (double)(N - 1) / (double)N * std::max(1.0, 1.0 + prm->diff_rot);
    s->amax = std::max(std::fabs(host_dshift(vmax, prm->doppler_mode)), std::fabs(host_dshift(-vmax, prm->doppler_mode)));

    SOAP_CUDA(s, s->d_mu.reserve(ncell));
    SOAP_CUDA(s, s->d_w.reserve(ncell));
    SOAP_CUDA(s, s->d_vel.reserve(ncell));
    SOAP_CUDA(s, s->d_bin.reserve(ncell));
    SOAP_CUDA(s, s->d_col_a.reserve(N));
    SOAP_CUDA(s, s->d_Wbin.reserve((size_t)N * n_mu));
    SOAP_CUDA(s, s->d_col_sumw.reserve(N));
    SOAP_CUDA(s, s->d_col_nvis.reserve(N));
    SOAP_CUDA(s, s->d_colcnt.reserve((size_t)N * n_mu));
    SOAP_CUDA(s, s->d_cellpos.reserve((size_t)N * n_mu));
    SOAP_CUDA(s, s->d_row_start.reserve(n_mu + 1));
    SOAP_CUDA(s, s->d_info.reserve(1));
    const size_t ent_cap = std::max(s->cell_entries ? ncell : (size_t)0, (size_t)N * n_mu) + 2 * (size_t)n_mu + 8;
    SOAP_CUDA(s, s->d_ent32.reserve(ent_cap));
    SOAP_CUDA(s, s->d_ent64.reserve(ent_cap));
    s->comp_stride = 0;
    if (s->form_used == SOAP_FORM_COMPOSITE) {
        s->comp_stride = round_up4(n_mu);
        SOAP_CUDA(s, s->d_cWp.reserve((size_t)((N + 1) / 2) * s->comp_stride));
        SOAP_CUDA(s, s->d_chdr.reserve((size_t)(N + 1) / 2 + 1));
    }

    if (!s->d_geom_done.ptr) {
        SOAP_CUDA(s, s->d_geom_done.reserve(1));
        SOAP_CUDA(s, cudaMemsetAsync(s->d_geom_done.ptr, 0, sizeof(unsigned int), st));  // once per handle
    }
    MuCentres mc{};
    for (int b = 0; b < n_mu; ++b) mc.v[b] = prm->mu_centres[b];
    Rotation rot{prm->vsini_kms, sini, cosi, prm->diff_rot};
    // a1 + a2 in one launch: the last CTA compacts the binned weights into the entry list - from a shared-memory copy of
    // the binned weights when they fit (geometry.cuh, finalize_columns_smem)
    const size_t fin_bytes = fin_smem_bytes(N, n_mu);
    const bool fin_smem = fin_bytes <= kFinSmemMax;
    if (fin_smem && !s->attr_geom_set) {
        SOAP_CUDA(s, cudaFuncSetAttribute(geometry_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFinSmemMax));
        s->attr_geom_set = true;
    }
    ga = GeomArgs{};
    ga.N = N;
    ga.mode = prm->doppler_mode;
    ga.n_mu = n_mu;
    ga.cells = s->cell_entries ? 1 : 0;
    ga.comp_stride = s->comp_stride;
    ga.fin_smem = fin_smem ? 1 : 0;
    ga.n_ctas = (N + geom_cols_per_cta(N) - 1) / geom_cols_per_cta(N);
    ga.rot = rot;
    ga.u1 = prm->ld_u1;
    ga.u2 = prm->ld_u2;
    ga.mu_centres = mc;
    ga.mu_out = s->d_mu.ptr;
    ga.w_out = s->d_w.ptr;
    ga.vel_out = s->d_vel.ptr;
    ga.bin_out = s->d_bin.ptr;
    ga.col_a = s->d_col_a.ptr;
    ga.Wbin = s->d_Wbin.ptr;
    ga.col_sumw = s->d_col_sumw.ptr;
    ga.col_nvis = s->d_col_nvis.ptr;
    ga.ent32 = s->d_ent32.ptr;
    ga.ent64 = s->d_ent64.ptr;
    ga.row_start = s->d_row_start.ptr;
    ga.info = s->d_info.ptr;
    ga.done = s->d_geom_done.ptr;
    ga.colcnt = s->d_colcnt.ptr;
    ga.cellpos = s->d_cellpos.ptr;
    ga.comp_Wp = s->comp_stride ? s->d_cWp.ptr : nullptr;
    ga.comp_hdr = s->d_chdr.ptr;
    fin_bytes_out = fin_smem ? fin_bytes : 0;
    return SOAP_OK;
}

static int geometry_finish(soap_star *s, cudaStream_t st, soap_geom_info *info) {
    const soap_star_params *prm = &s->prm;
    const int N = prm->grid_n, n_mu = prm->n_mu;
    if (s->cell_entries) {
        write_cell_entries_kernel<<<(N + kCellWarps - 1) / kCellWarps, 32 * kCellWarps, 0, st>>>(
            N, n_mu, prm->doppler_mode, s->d_vel.ptr, s->d_w.ptr, s->d_bin.ptr, s->d_cellpos.ptr, s->d_ent32.ptr, s->d_ent64.ptr);
        SOAP_LAUNCH_CHECK(s, "write_cell_entries_kernel");
    }
    s->ready = true;
    if (info) {
        DevInfo di;
        SOAP_CUDA(s, cudaMemcpyAsync(&di, s->d_info.ptr, sizeof(di), cudaMemcpyDeviceToHost, st));
        SOAP_CUDA(s, cudaStreamSynchronize(st));
        info->n_visible = di.n_visible;
        info->n_entries = s->cell_entries ? di.n_visible : di.n_entries;
        info->sum_weights = di.sum_weights;
        info->max_abs_dshift = di.max_abs_dshift;
    }
    return SOAP_OK;
}

int soap_disk_geometry(soap_star *s, const soap_star_params *prm, void *stream, soap_geom_info *info) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    int rc = geometry_check(s, prm);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    GeomArgs ga;
    size_t fin_bytes = 0;
    if ((rc = geometry_prepare(s, prm, st, ga, fin_bytes))) return rc;
    // a1 + a2 in one launch: the last CTA compacts the binned weights into the entry list
    geometry_kernel<<<ga.n_ctas, 32 * kGeomWarps, fin_bytes, st>>>(ga, nullptr, nullptr, 1);
    SOAP_LAUNCH_CHECK(s, "geometry_kernel");
    return geometry_finish(s, st, info);
}

// config 5: the geometry of many stars in ONE launch (every star's CTAs side by side, each star with its own last-CTA
// finalisation); per-cell entry lists (differential rotation) are written by one more launch per such star.
int soap_batch_disk_geometry(soap_star *const *stars, int32_t n_stars, const soap_star_params *const *params, void *stream,
                             soap_geom_info *infos) {
    if (!stars || !params || n_stars < 0) return SOAP_ERR_INVALID_ARG;
    for (int k = 0; k < n_stars; ++k)
        if (!stars[k]) return SOAP_ERR_INVALID_ARG;
    if (n_stars == 0) return SOAP_OK;
    soap_star *s0 = stars[0];
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    bool one_launch = n_stars > 1;
    for (int k = 0; k < n_stars; ++k) {  // every argument of every star is checked before anything is enqueued
        int rc = geometry_check(stars[k], params[k]);
        if (rc) return rc;
        for (int j = 0; j < k; ++j)
            if (stars[j] == stars[k]) return stars[k]->fail(SOAP_ERR_INVALID_ARG, "star %d appears twice in the batch", k);
        one_launch = one_launch && stars[k]->device == s0->device;
    }
    if (!one_launch) {  // a single star, or several devices: per-star calls
        for (int k = 0; k < n_stars; ++k) {
            int rc = soap_disk_geometry(stars[k], params[k], stream, infos ? infos + k : nullptr);
            if (rc) return rc;
        }
        return SOAP_OK;
    }
    std::vector<GeomArgs> args((size_t)n_stars);
    std::vector<int> cta0((size_t)n_stars + 1);
    size_t fin_bytes = 0;
    int total = 0;
    for (int k = 0; k < n_stars; ++k) {
        size_t fb = 0;
        int rc = geometry_prepare(stars[k], params[k], st, args[k], fb);
        if (rc) return rc;
        fin_bytes = std::max(fin_bytes, fb);
        cta0[k] = total;
        total += args[k].n_ctas;
    }
    cta0[n_stars] = total;
    const size_t a_bytes = (size_t)n_stars * sizeof(GeomArgs), c_off = (a_bytes + 15) & ~(size_t)15;
    const size_t bytes = c_off + (size_t)(n_stars + 1) * sizeof(int);
    if (bytes > s0->d_gargs.cap) {
        SOAP_CUDA(s0, cudaStreamSynchronize(st));  // an earlier launch may still read the old buffer
        SOAP_CUDA(s0, s0->d_gargs.reserve(bytes + 4096));
    }
    // pageable sources: the runtime stages them before returning, so the vectors may go out of scope
    SOAP_CUDA(s0, cudaMemcpyAsync(s0->d_gargs.ptr, args.data(), a_bytes, cudaMemcpyHostToDevice, st));
    SOAP_CUDA(s0, cudaMemcpyAsync(s0->d_gargs.ptr + c_off, cta0.data(), (size_t)(n_stars + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    geometry_kernel<<<total, 32 * kGeomWarps, fin_bytes, st>>>(args[0], reinterpret_cast<const GeomArgs *>(s0->d_gargs.ptr),
                                                            reinterpret_cast<const int *>(s0->d_gargs.ptr + c_off), n_stars);
    SOAP_LAUNCH_CHECK(s0, "geometry_kernel");
    for (int k = 0; k < n_stars; ++k) {
        int rc = geometry_finish(stars[k], st, infos ? infos + k : nullptr);
        if (rc) return rc;
    }
    return SOAP_OK;
}

int soap_integrate_quiet(soap_star *s, const soap_spectra *quiet, void *out, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!s->ready) return s->fail(SOAP_ERR_NOT_READY, "soap_disk_geometry has not been called");
    int rc = check_spectra(s, quiet, "quiet");
    if (rc) return rc;
    if (!out) return s->fail(SOAP_ERR_INVALID_ARG, "out is NULL");
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return quiet->dtype == SOAP_F32 ? quiet_impl<float>(s, quiet, out, st) : quiet_impl<double>(s, quiet, out, st);
}

int soap_integrate_quiet_static(soap_star *s, const soap_spectra *quiet, void *out, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!s->ready) return s->fail(SOAP_ERR_NOT_READY, "soap_disk_geometry has not been called");
    int rc = check_spectra(s, quiet, "quiet");
    if (rc) return rc;
    if (!out) return s->fail(SOAP_ERR_INVALID_ARG, "out is NULL");
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return quiet->dtype == SOAP_F32 ? quiet_static_impl<float>(s, quiet, out, st) : quiet_static_impl<double>(s, quiet, out, st);
}

int soap_active_timeseries_evolving(soap_star *s, const soap_spectra *quiet, const soap_spectra *spot,
                                    const soap_spectra *facula, const soap_region *regions, int32_t n_regions,
                                    const double *phases, int32_t n_phases, const double *radii, void *out_total,
                                    void *out_flux, void *out_cb, int64_t out_pitch, int32_t *n_active, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!s->ready) return s->fail(SOAP_ERR_NOT_READY, "soap_disk_geometry has not been called");
    int rc = check_spectra(s, quiet, "quiet");
    if (rc) return rc;
    if (spot && ((rc = check_spectra(s, spot, "spot")) || (rc = check_same_grid(s, quiet, spot, "spot")))) return rc;
    if (facula && ((rc = check_spectra(s, facula, "facula")) || (rc = check_same_grid(s, quiet, facula, "facula")))) return rc;
    if ((rc = check_regions(s, regions, n_regions, phases, n_phases, spot, facula))) return rc;
    if (radii)
        for (size_t k = 0; k < (size_t)n_phases * (size_t)n_regions; ++k)
            if (!(radii[k] < 1.0) || !std::isfinite(radii[k])) return s->fail(SOAP_ERR_INVALID_ARG, "radii[%zu] must be finite and < 1", k);
    if (n_phases == 0) return SOAP_OK;
    if (!out_total && !out_flux && !out_cb) return s->fail(SOAP_ERR_INVALID_ARG, "every output is NULL");
    if (out_pitch < quiet->n_pix) return s->fail(SOAP_ERR_INVALID_ARG, "out_pitch must be >= n_pix");
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool one_launch_path = quiet->dtype == SOAP_F32 && s->prm.diff_rot == 0.0;
    if (!one_launch_path && !s->reuse_lists && !s->regions_uploaded &&
        (rc = upload_region_centres(s, regions, n_regions, phases, n_phases, radii, st)))
        return rc;
    // Two or three outputs of a solid-body fp32 star: ONE map and ONE shift-interpolate-accumulate pass (effects launch,
    // sia_f32.cuh) unless SOAP_OPT_EFFECT_PASSES asks for a pass per effect or the wider map does not fit in shared memory.
    const int n_out = (out_total ? 1 : 0) + (out_flux ? 1 : 0) + (out_cb ? 1 : 0);
    if (one_launch_path && n_out >= 2 && !s->reuse_lists && !s->opt_effect_passes) {
        const int N = s->prm.grid_n, kinds = effect_kinds(kEffectAll, spot, facula);
        if (prep_smem_bytes(s->prm.n_mu, std::max(32, (N + kPrepCluster - 1) / kPrepCluster), N, n_regions, kinds) <= 200 * 1024) {
            ActiveCall c{s, quiet, spot, facula, regions, n_regions, phases, n_phases, radii, out_total, out_pitch, out_flux, out_cb};
            if ((rc = active_f32_launch(&c, 1, kEffectAll, true, false, st))) return rc;
            if (n_active) {
                SOAP_CUDA(s, cudaMemcpyAsync(n_active, s->d_nactive.ptr, (size_t)n_phases * sizeof(int), cudaMemcpyDeviceToHost, st));
                SOAP_CUDA(s, cudaStreamSynchronize(st));
                long long tot = 0;
                for (int p = 0; p < n_phases; ++p) tot += n_active[p];
                s->last_active_cells = tot;
            }
            return SOAP_OK;
        }
    }
    // total and flux-only share the entry lists (weights w LB_t(mu)); CB-only needs the plain weights w, which
    // are the same lists again when both limb-brightening laws are identically 1
    const bool lb_one = lb_is_one(spot) && lb_is_one(facula);
    struct Pass { int effect; void *out; } passes[3] = {{SOAP_EFFECT_TOTAL, out_total}, {SOAP_EFFECT_FLUX, out_flux}, {SOAP_EFFECT_CB, out_cb}};
    bool have_lb_lists = s->reuse_lists;
    for (const Pass &ps : passes) {
        if (!ps.out) continue;
        const bool prepare = ps.effect == SOAP_EFFECT_CB ? !(have_lb_lists && lb_one) : !have_lb_lists;
        if (one_launch_path) {
            ActiveCall c{s, quiet, spot, facula, regions, n_regions, phases, n_phases, radii, ps.out, out_pitch};
            rc = active_f32_launch(&c, 1, ps.effect, prepare, false, st);
            if (rc) return rc;
            if (ps.effect != SOAP_EFFECT_CB) have_lb_lists = true;
            continue;
        }
        rc = quiet->dtype == SOAP_F32
                 ? active_impl<float>(s, quiet, spot, facula, n_regions, n_phases, ps.effect, prepare, ps.out, out_pitch, st)
                 : active_impl<double>(s, quiet, spot, facula, n_regions, n_phases, ps.effect, prepare, ps.out, out_pitch, st);
        if (rc) return rc;
        if (ps.effect != SOAP_EFFECT_CB) have_lb_lists = true;
    }
    if (n_active) {
        SOAP_CUDA(s, cudaMemcpyAsync(n_active, s->d_nactive.ptr, (size_t)n_phases * sizeof(int), cudaMemcpyDeviceToHost, st));
        SOAP_CUDA(s, cudaStreamSynchronize(st));
        long long tot = 0;
        for (int p = 0; p < n_phases; ++p) tot += n_active[p];
        s->last_active_cells = tot;
    }
    return SOAP_OK;
}

int soap_active_timeseries_effects(soap_star *s, const soap_spectra *quiet, const soap_spectra *spot,
                                   const soap_spectra *facula, const soap_region *regions, int32_t n_regions,
                                   const double *phases, int32_t n_phases, void *out_total, void *out_flux, void *out_cb,
                                   int64_t out_pitch, int32_t *n_active, void *stream) {
    return soap_active_timeseries_evolving(s, quiet, spot, facula, regions, n_regions, phases, n_phases, nullptr, out_total,
                                           out_flux, out_cb, out_pitch, n_active, stream);
}

int soap_active_timeseries(soap_star *s, const soap_spectra *quiet, const soap_spectra *spot, const soap_spectra *facula,
                           const soap_region *regions, int32_t n_regions, const double *phases, int32_t n_phases,
                           void *out_delta, int64_t out_pitch, int32_t *n_active, void *stream) {
    if (s && s->ready && n_phases > 0 && !out_delta) return s->fail(SOAP_ERR_INVALID_ARG, "out_delta is NULL");
    return soap_active_timeseries_effects(s, quiet, spot, facula, regions, n_regions, phases, n_phases, out_delta, nullptr,
                                          nullptr, out_pitch, n_active, stream);
}

int soap_lower_resolution(soap_star *s, const void *in, int64_t n_rows, int64_t n_pix, int64_t in_pitch, int32_t dtype,
                          double lambda0, double dlambda, double resolution, void *out, int64_t out_pitch, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!in || !out) return s->fail(SOAP_ERR_INVALID_ARG, "in / out is NULL");
    if (in == out) return s->fail(SOAP_ERR_INVALID_ARG, "in-place resolution lowering is not supported");
    if (n_rows < 0 || n_pix < 1 || in_pitch < n_pix || out_pitch < n_pix) return s->fail(SOAP_ERR_INVALID_ARG, "bad n_rows / n_pix / pitch");
    if (dtype != SOAP_F32 && dtype != SOAP_F64) return s->fail(SOAP_ERR_INVALID_ARG, "unknown dtype %d", dtype);
    if (!(dlambda > 0.0) || !(lambda0 > 0.0) || !std::isfinite(dlambda) || !std::isfinite(lambda0))
        return s->fail(SOAP_ERR_INVALID_ARG, "lambda0 and dlambda must be positive and finite");
    if (!(resolution > 0.0) || !std::isfinite(resolution)) return s->fail(SOAP_ERR_INVALID_ARG, "resolution must be positive and finite");
    if (n_rows == 0) return SOAP_OK;
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    LsfArgs a{};
    a.in = in;
    a.out = out;
    a.n_rows = n_rows;
    a.n_pix = n_pix;
    a.in_pitch = in_pitch;
    a.out_pitch = out_pitch;
    a.lambda0 = lambda0;
    a.k = dlambda;
    a.R = resolution;
    a.fwhm_to_sigma = 1.0 / (2.0 * std::sqrt(2.0 * std::log(2.0)));
    const double lam_last = lambda0 + dlambda * (double)(n_pix - 1);
    const double j_last = std::ceil(kLsfNsig * (lam_last / resolution * a.fwhm_to_sigma) / dlambda);
    if (j_last > (double)kLsfMaxJ)
        return s->fail(SOAP_ERR_UNSUPPORTED, "line-spread function of %.0f pixels half-width exceeds %d", j_last, kLsfMaxJ);
    a.J_max = (int)j_last;
    {
        // the steps of J(m) = ceil(5 sigma_m / k) (non-decreasing: every operation is monotone), by bisection on the defining
        // expression - the operations, and so the results, of the kernels' per-pixel evaluation
        auto jm = [&](long long m) {
            volatile double t = dlambda * (double)m;  // (no contraction into an FMA)
            const double lam = lambda0 + t;
            volatile double sg = lam / resolution;
            volatile double sigma = sg * a.fwhm_to_sigma;
            volatile double five = kLsfNsig * sigma;
            return (int)std::ceil(five / dlambda);
        };
        a.jm0 = jm(0);
        a.n_breaks = 0;
        const int j_end = jm(n_pix - 1);
        // (the table serves the row-pair kernel, J <= 16: at most 16 steps; wider functions never read it)
        for (int J = a.jm0 + 1; J <= j_end && a.n_breaks < kLsfBreaks; ++J) {
            long long lo = 0, hi = n_pix - 1;  // jm(lo) < J <= jm(hi)
            while (hi - lo > 1) {
                const long long mid = lo + (hi - lo) / 2;
                if (jm(mid) >= J) hi = mid;
                else lo = mid;
            }
            a.jm_break[a.n_breaks++] = hi;
        }
        const double kr = dlambda * resolution / a.fwhm_to_sigma;
        a.h_scale = 0.5 * kr * kr;
    }
    const size_t elem = dtype == SOAP_F64 ? 8 : 4;
    const size_t smem = lsf_smem_bytes(a.J_max, elem);
    const unsigned tiles = (unsigned)((n_pix + kLsfThreads - 1) / kLsfThreads);
    // tiles x row groups, at least ~4 waves of CTAs so that the last wave is short; a CTA keeps its weights for all
    // the rows of its group
    unsigned gy = (unsigned)std::max<long long>(1, std::min<long long>(n_rows, ((long long)s->n_sm * 8 * 4 + tiles - 1) / tiles));
    // fp32 with 16-byte aligned rows: the register-window kernel, persistent CTAs over (tile, row) items
    const bool aligned = !(in_pitch & 3) && !(out_pitch & 3) && !(reinterpret_cast<uintptr_t>(in) & 15) &&
                         !(reinterpret_cast<uintptr_t>(out) & 15);
    if (dtype == SOAP_F32 && aligned && a.J_max <= 24) {
        auto launch = [&](auto kern, size_t vsmem) -> int {
            SOAP_CUDA(s, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)vsmem));
            int occ = 0;
            SOAP_CUDA(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kLsfThreads, vsmem));
            if (occ < 1) return s->fail(SOAP_ERR_UNSUPPORTED, "resolution-lowering kernel does not fit on an SM");
            const long long items = ((n_pix + kLsfTileV - 1) / kLsfTileV) * n_rows;
            const unsigned g = (unsigned)std::max<long long>(1, std::min<long long>(items, (long long)s->n_sm * occ));
            kern<<<g, kLsfThreads, vsmem, st>>>(a);
            return SOAP_OK;
        };
        auto launch_p = [&](auto kern, size_t psmem) -> int {  // rows in pairs (lsf.cuh, lower_resolution_p_kernel)
            SOAP_CUDA(s, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psmem));
            int occ = 0;
            SOAP_CUDA(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kLsfThreads, psmem));
            if (occ < 1) return s->fail(SOAP_ERR_UNSUPPORTED, "resolution-lowering kernel does not fit on an SM");
            const long long items = ((n_pix + kLsfTileP - 1) / kLsfTileP) * ((n_rows + 1) / 2);
            const unsigned g = (unsigned)std::max<long long>(1, std::min<long long>(items, (long long)s->n_sm * occ));
            kern<<<g, kLsfThreads, psmem, st>>>(a);
            return SOAP_OK;
        };
        int rc;
        if (a.J_max <= 16) {
            if (a.J_max <= 4) rc = launch_p(lower_resolution_p_kernel<4>, lsf_p_smem_bytes<4>());
            else if (a.J_max <= 8) rc = launch_p(lower_resolution_p_kernel<8>, lsf_p_smem_bytes<8>());
            else if (a.J_max <= 12) rc = launch_p(lower_resolution_p_kernel<12>, lsf_p_smem_bytes<12>());
            else if (a.J_max <= 14) rc = launch_p(lower_resolution_p_kernel<14>, lsf_p_smem_bytes<14>());
            else rc = launch_p(lower_resolution_p_kernel<16>, lsf_p_smem_bytes<16>());
            if (rc) return rc;
            SOAP_LAUNCH_CHECK(s, "lower_resolution_p_kernel");
            return SOAP_OK;
        }
        if (a.J_max <= 4) rc = launch(lower_resolution_v_kernel<4>, lsf_v_smem_bytes<4>());
        else if (a.J_max <= 8) rc = launch(lower_resolution_v_kernel<8>, lsf_v_smem_bytes<8>());
        else if (a.J_max <= 12) rc = launch(lower_resolution_v_kernel<12>, lsf_v_smem_bytes<12>());
        else if (a.J_max <= 16) rc = launch(lower_resolution_v_kernel<16>, lsf_v_smem_bytes<16>());
        else if (a.J_max <= 20) rc = launch(lower_resolution_v_kernel<20>, lsf_v_smem_bytes<20>());
        else rc = launch(lower_resolution_v_kernel<24>, lsf_v_smem_bytes<24>());
        if (rc) return rc;
        SOAP_LAUNCH_CHECK(s, "lower_resolution_v_kernel");
        return SOAP_OK;
    }
    if (dtype == SOAP_F32) {
        SOAP_CUDA(s, cudaFuncSetAttribute(lower_resolution_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        lower_resolution_kernel<float><<<dim3(tiles, gy), kLsfThreads, smem, st>>>(a);
    } else {
        SOAP_CUDA(s, cudaFuncSetAttribute(lower_resolution_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        lower_resolution_kernel<double><<<dim3(tiles, gy), kLsfThreads, smem, st>>>(a);
    }
    SOAP_LAUNCH_CHECK(s, "lower_resolution_kernel");
    return SOAP_OK;
}

int soap_line_rvs(soap_star *s, const void *rows, int64_t n_rows, int64_t n_pix, int64_t pitch, int32_t dtype, double lambda0,
                  double dlambda, const double *centres, const double *half_widths, int64_t n_lines, const double *norm,
                  int64_t edge, double *out_rv, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!rows || !centres || !half_widths || !norm || !out_rv) return s->fail(SOAP_ERR_INVALID_ARG, "NULL argument");
    if (n_rows < 0 || n_lines < 0 || n_pix < 1 || pitch < n_pix || edge < 0) return s->fail(SOAP_ERR_INVALID_ARG, "bad sizes");
    if (dtype != SOAP_F32 && dtype != SOAP_F64) return s->fail(SOAP_ERR_INVALID_ARG, "unknown dtype %d", dtype);
    if (!(dlambda > 0.0) || !std::isfinite(dlambda) || !std::isfinite(lambda0)) return s->fail(SOAP_ERR_INVALID_ARG, "bad wavelength grid");
    if (n_rows == 0 || n_lines == 0) return SOAP_OK;
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    RvArgs a{};
    a.rows = rows;
    a.n_rows = n_rows;
    a.n_pix = n_pix;
    a.pitch = pitch;
    a.lambda0 = lambda0;
    a.k = dlambda;
    a.centres = centres;
    a.half_widths = half_widths;
    a.norm = norm;
    a.n_lines = n_lines;
    a.edge = edge;
    a.rv = out_rv;
    a.rows_pass = (int)std::min<long long>(kRvRows, n_rows);
    const unsigned gx = (unsigned)((n_lines + kRvWarps - 1) / kRvWarps);
    const unsigned gy = (unsigned)std::min<long long>((n_rows + a.rows_pass - 1) / a.rows_pass, 65535);  // one warp per (line, rows_pass rows)
    if (!s->attr_rv_set) {
        SOAP_CUDA(s, cudaFuncSetAttribute(line_rv_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rv_smem_bytes<float>(kRvRows)));
        SOAP_CUDA(s, cudaFuncSetAttribute(line_rv_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rv_smem_bytes<double>(kRvRows)));
        s->attr_rv_set = true;
    }
    if (dtype == SOAP_F32) line_rv_kernel<float><<<dim3(gx, gy), 32 * kRvWarps, rv_smem_bytes<float>(a.rows_pass), st>>>(a);
    else line_rv_kernel<double><<<dim3(gx, gy), 32 * kRvWarps, rv_smem_bytes<double>(a.rows_pass), st>>>(a);
    SOAP_LAUNCH_CHECK(s, "line_rv_kernel");
    return SOAP_OK;
}

int soap_contrast_planck(soap_star *s, double lambda0, double dlambda, int64_t n_pix, double t_quiet, double t_active, void *out,
                         int32_t dtype, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!out) return s->fail(SOAP_ERR_INVALID_ARG, "out is NULL");
    if (n_pix < 0 || n_pix > (1LL << 40)) return s->fail(SOAP_ERR_INVALID_ARG, "bad n_pix");
    if (dtype != SOAP_F32 && dtype != SOAP_F64) return s->fail(SOAP_ERR_INVALID_ARG, "unknown dtype %d", dtype);
    if (!(dlambda > 0.0) || !(lambda0 > 0.0) || !std::isfinite(dlambda) || !std::isfinite(lambda0))
        return s->fail(SOAP_ERR_INVALID_ARG, "lambda0 and dlambda must be positive and finite");
    if (!(t_quiet > 0.0) || !(t_active > 0.0) || !std::isfinite(t_quiet) || !std::isfinite(t_active))
        return s->fail(SOAP_ERR_INVALID_ARG, "temperatures must be positive and finite");
    if (n_pix == 0) return SOAP_OK;
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)((n_pix + 255) / 256);
    if (dtype == SOAP_F32)
        contrast_planck_kernel<float><<<grid, 256, 0, st>>>(lambda0, dlambda, n_pix, 1.0 / t_quiet, 1.0 / t_active, static_cast<float *>(out));
    else
        contrast_planck_kernel<double><<<grid, 256, 0, st>>>(lambda0, dlambda, n_pix, 1.0 / t_quiet, 1.0 / t_active, static_cast<double *>(out));
    SOAP_LAUNCH_CHECK(s, "contrast_planck_kernel");
    return SOAP_OK;
}

int soap_get_stats(soap_star *s, soap_stats *stats, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!stats) return s->fail(SOAP_ERR_INVALID_ARG, "stats is NULL");
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::memset(stats, 0, sizeof(*stats));
    if (s->ready) {
        DevInfo di;
        SOAP_CUDA(s, cudaMemcpyAsync(&di, s->d_info.ptr, sizeof(di), cudaMemcpyDeviceToHost, st));
        SOAP_CUDA(s, cudaStreamSynchronize(st));
        stats->quiet_entries = s->cell_entries ? di.n_visible : di.n_entries;
    }
    if (s->d_counters.ptr && s->d_sched.ptr && s->last_n_phases > 0) {
        ActiveCounters c;
        std::vector<int> work((size_t)s->last_n_phases);
        SOAP_CUDA(s, cudaMemcpyAsync(&c, s->d_counters.ptr, sizeof(c), cudaMemcpyDeviceToHost, st));
        SOAP_CUDA(s, cudaMemcpyAsync(work.data(), s->d_sched.ptr + s->last_n_phases, work.size() * sizeof(int), cudaMemcpyDeviceToHost, st));
        SOAP_CUDA(s, cudaStreamSynchronize(st));
        if (c.overflow) return s->fail(SOAP_ERR_CUDA, "active map: a phase's entry pool overflowed (the result of the last call is incomplete)");
        long long total = 0;
        for (int w : work) total += w;
        stats->active_entries = total;  // pad entries not counted
    }
    stats->active_cells = s->last_active_cells;
    stats->quiet_splits = s->last_quiet_splits;
    stats->tile_px = s->last_tile_px;
    stats->form = s->last_form ? s->last_form : s->form_used;
    stats->launches = s->launches;
    if (s->opt_timing) {
        SOAP_CUDA(s, cudaStreamSynchronize(st));
        if (s->ev_valid[0]) SOAP_CUDA(s, cudaEventElapsedTime(&stats->quiet_kernel_ms, s->ev[0], s->ev[1]));
        if (s->ev_valid[1]) SOAP_CUDA(s, cudaEventElapsedTime(&stats->active_kernel_ms, s->ev[2], s->ev[3]));
    }
    return SOAP_OK;
}

int soap_export_geometry(soap_star *s, double *mu, double *vel, double *w, int32_t *bin) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!s->ready) return s->fail(SOAP_ERR_NOT_READY, "soap_disk_geometry has not been called");
    SOAP_CUDA(s, cudaSetDevice(s->device));
    SOAP_CUDA(s, cudaDeviceSynchronize());
    const size_t ncell = (size_t)s->prm.grid_n * s->prm.grid_n;
    if (mu) SOAP_CUDA(s, cudaMemcpy(mu, s->d_mu.ptr, ncell * sizeof(double), cudaMemcpyDeviceToHost));
    if (vel) SOAP_CUDA(s, cudaMemcpy(vel, s->d_vel.ptr, ncell * sizeof(double), cudaMemcpyDeviceToHost));
    if (w) SOAP_CUDA(s, cudaMemcpy(w, s->d_w.ptr, ncell * sizeof(double), cudaMemcpyDeviceToHost));
    if (bin) SOAP_CUDA(s, cudaMemcpy(bin, s->d_bin.ptr, ncell * sizeof(int), cudaMemcpyDeviceToHost));
    return SOAP_OK;
}

int soap_synthesize_host(soap_star *s, const soap_star_params *prm, const soap_spectra *quiet, const soap_spectra *spot,
                         const soap_spectra *facula, const soap_region *regions, int32_t n_regions, const double *phases,
                         int32_t n_phases, void *out_quiet, void *out_delta, int32_t *n_active, void *stream) {
    if (!s) return SOAP_ERR_INVALID_ARG;
    if (!quiet || !quiet->data) return s->fail(SOAP_ERR_INVALID_ARG, "quiet spectra missing");
    if (!out_quiet) return s->fail(SOAP_ERR_INVALID_ARG, "out_quiet is NULL");
    if (n_phases > 0 && !out_delta) return s->fail(SOAP_ERR_INVALID_ARG, "out_delta is NULL");
    SOAP_CUDA(s, cudaSetDevice(s->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (prm && quiet->dtype == SOAP_F32 && n_phases > 0 && quiet->n_pix >= 16LL * f32::kTile && prm->n_mu >= 1 &&
        prm->n_mu <= SOAP_MAX_MU && quiet->pitch >= quiet->n_pix && !(quiet->pitch & 3))
        return synthesize_host_pipelined(s, prm, quiet, spot, facula, regions, n_regions, phases, n_phases, out_quiet, out_delta,
                                         n_active, st);
    const soap_spectra *in[3] = {quiet, spot, facula};
    soap_spectra dev[3];
    const size_t esz = quiet->dtype == SOAP_F64 ? 8 : 4;
    if (!prm) return s->fail(SOAP_ERR_INVALID_ARG, "params is NULL");
    if (prm->n_mu < 1 || prm->n_mu > SOAP_MAX_MU) return s->fail(SOAP_ERR_INVALID_ARG, "n_mu must be in 1..%d", SOAP_MAX_MU);
    for (int k = 0; k < 3; ++k) {
        if (!in[k]) continue;
        if (!in[k]->data) return s->fail(SOAP_ERR_INVALID_ARG, "spectra %d: data is NULL", k);
        if (in[k]->n_pix < 2 || in[k]->pitch < in[k]->n_pix || (in[k]->pitch & 3) || in[k]->dtype != quiet->dtype)
            return s->fail(SOAP_ERR_INVALID_ARG, "spectra %d: bad n_pix / pitch / dtype", k);
        const size_t bytes = (size_t)prm->n_mu * in[k]->pitch * esz;
        SOAP_CUDA(s, s->d_stage[k].reserve(bytes));
        SOAP_CUDA(s, cudaMemcpyAsync(s->d_stage[k].ptr, in[k]->data, bytes, cudaMemcpyHostToDevice, st));
        dev[k] = *in[k];
        dev[k].data = s->d_stage[k].ptr;
        if (k > 0 && in[k]->contrast) {
            SOAP_CUDA(s, s->d_stage_c[k].reserve((size_t)in[k]->n_pix * esz));
            SOAP_CUDA(s, cudaMemcpyAsync(s->d_stage_c[k].ptr, in[k]->contrast, (size_t)in[k]->n_pix * esz, cudaMemcpyHostToDevice, st));
            dev[k].contrast = s->d_stage_c[k].ptr;
        } else {
            dev[k].contrast = nullptr;
        }
    }
    const long long P = quiet->n_pix;
    SOAP_CUDA(s, s->d_out_q.reserve((size_t)P * esz));
    if (n_phases > 0) SOAP_CUDA(s, s->d_out_d.reserve((size_t)n_phases * P * esz));
    int rc = soap_disk_geometry(s, prm, stream, nullptr);
    if (rc) return rc;
    if ((rc = soap_integrate_quiet(s, &dev[0], s->d_out_q.ptr, stream))) return rc;
    if (n_phases > 0) {
        rc = soap_active_timeseries(s, &dev[0], spot ? &dev[1] : nullptr, facula ? &dev[2] : nullptr, regions, n_regions, phases,
                                    n_phases, s->d_out_d.ptr, P, nullptr, stream);
        if (rc) return rc;
        SOAP_CUDA(s, cudaMemcpyAsync(out_delta, s->d_out_d.ptr, (size_t)n_phases * P * esz, cudaMemcpyDeviceToHost, st));
        if (n_active)
            SOAP_CUDA(s, cudaMemcpyAsync(n_active, s->d_nactive.ptr, (size_t)n_phases * sizeof(int), cudaMemcpyDeviceToHost, st));
    }
    SOAP_CUDA(s, cudaMemcpyAsync(out_quiet, s->d_out_q.ptr, (size_t)P * esz, cudaMemcpyDeviceToHost, st));
    SOAP_CUDA(s, cudaStreamSynchronize(st));
    return SOAP_OK;
}

// Batch entry points (config 5): the stars are independent, so their work is dealt round-robin to three lanes - the
// caller's stream and two side streams of the first handle, forked from and joined back into the caller's stream with
// events.  Each star's big kernels fill the GPU on their own; what overlaps is the tail of one star's kernel with the
// start of the next star's, and the small kernels (active map) of one star with the big kernels of another.
static int batch_fork(soap_star *s0, cudaStream_t st, cudaStream_t lanes[3]) {
    SOAP_CUDA(s0, cudaSetDevice(s0->device));
    if (!s0->s_h2d) SOAP_CUDA(s0, cudaStreamCreateWithFlags(&s0->s_h2d, cudaStreamNonBlocking));
    if (!s0->s_d2h) SOAP_CUDA(s0, cudaStreamCreateWithFlags(&s0->s_d2h, cudaStreamNonBlocking));
    while (s0->ev_pipe.size() < 3) {
        cudaEvent_t e;
        SOAP_CUDA(s0, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        s0->ev_pipe.push_back(e);
    }
    lanes[0] = st;
    lanes[1] = s0->s_h2d;
    lanes[2] = s0->s_d2h;
    SOAP_CUDA(s0, cudaEventRecord(s0->ev_pipe[0], st));
    SOAP_CUDA(s0, cudaStreamWaitEvent(lanes[1], s0->ev_pipe[0], 0));
    SOAP_CUDA(s0, cudaStreamWaitEvent(lanes[2], s0->ev_pipe[0], 0));
    return SOAP_OK;
}
static int batch_join(soap_star *s0, cudaStream_t st, cudaStream_t lanes[3]) {
    for (int l = 1; l < 3; ++l) {
        SOAP_CUDA(s0, cudaEventRecord(s0->ev_pipe[l], lanes[l]));
        SOAP_CUDA(s0, cudaStreamWaitEvent(st, s0->ev_pipe[l], 0));
    }
    return SOAP_OK;
}

int soap_batch_integrate_quiet(soap_star *const *stars, int32_t n_stars, const soap_spectra *const *quiet, void *const *out,
                               void *stream) {
    if (!stars || !quiet || !out || n_stars < 0) return SOAP_ERR_INVALID_ARG;
    for (int k = 0; k < n_stars; ++k)
        if (!stars[k]) return SOAP_ERR_INVALID_ARG;
    if (n_stars == 0) return SOAP_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    soap_star *s0 = stars[0];
    // ---- every argument is checked before anything is enqueued ---------------------------------------------------------
    bool one_launch = true;
    for (int k = 0; k < n_stars; ++k) {
        soap_star *s = stars[k];
        if (!s->ready) return s->fail(SOAP_ERR_NOT_READY, "soap_disk_geometry has not been called (star %d of the batch)", k);
        int rc = check_spectra(s, quiet[k], "quiet");
        if (rc) return rc;
        if (!out[k]) return s->fail(SOAP_ERR_INVALID_ARG, "out is NULL (star %d of the batch)", k);
        for (int j = 0; j < k; ++j)
            if (stars[j] == s) return s->fail(SOAP_ERR_INVALID_ARG, "star %d appears twice in the batch", k);
        one_launch = one_launch && s->device == s0->device && composite_applies(s, quiet[k]) && s->comp_stride == s0->comp_stride;
    }
    SOAP_CUDA(s0, cudaSetDevice(s0->device));
    // a launch sizes its shared memory for the largest pair table AND the largest halo among its stars: a group that mixes
    // a fine grid with a fast rotator may not fit although each star does on its own - such a batch takes the per-star lanes
    for (int k0 = 0; one_launch && k0 < n_stars; k0 += comp::kMaxStars) {
        int max_pairs = 0, max_halo = 0;
        for (int k = k0; k < std::min(n_stars, k0 + comp::kMaxStars); ++k) {
            max_pairs = std::max(max_pairs, (stars[k]->prm.grid_n + 1) / 2);
            max_halo = std::max(max_halo, halo_for(stars[k], quiet[k]));
        }
        one_launch = comp::smem_bytes(s0->comp_stride, max_pairs, max_halo) <= (size_t)200 * 1024 / comp::kCtasPerSm;
    }
    if (one_launch) {
        // the composite-column kernel walks the flattened (star, tile, column pair) list: ONE launch for the batch
        // (groups of comp::kMaxStars stars when the batch is larger)
        for (int k0 = 0; k0 < n_stars; k0 += comp::kMaxStars) {
            const int n = std::min(comp::kMaxStars, n_stars - k0);
            std::vector<comp::Star> hs((size_t)n);
            int max_pairs = 0, max_mu = 0;
            for (int k = 0; k < n; ++k) {
                soap_star *s = stars[k0 + k];
                composite_fill(s, quiet[k0 + k], out[k0 + k], hs[k]);
                int rc = reserve_tickets(s, (size_t)hs[k].n_tiles + 1, st);
                if (rc) return rc;
                hs[k].ticket = s->d_tile_ticket.ptr;
                max_pairs = std::max(max_pairs, hs[k].n_pairs);
                max_mu = std::max(max_mu, s->prm.n_mu);
                s->last_tile_px = hs[k].L;
                s->last_form = SOAP_FORM_COMPOSITE;
            }
            if (n > 1) {
                if ((size_t)n > s0->d_cstars.cap) {
                    SOAP_CUDA(s0, cudaStreamSynchronize(st));  // an earlier launch may still read the old buffer
                    SOAP_CUDA(s0, s0->d_cstars.reserve((size_t)std::max(n, 64)));
                }
                // pageable source: the runtime stages it before returning, so `hs` may go out of scope
                SOAP_CUDA(s0, cudaMemcpyAsync(s0->d_cstars.ptr, hs.data(), (size_t)n * sizeof(comp::Star), cudaMemcpyHostToDevice, st));
            }
            int rc = launch_composite(s0, hs.data(), s0->d_cstars.ptr, n, s0->comp_stride, max_pairs, max_mu, st);
            if (rc) return rc;
        }
        return SOAP_OK;
    }
    // mixed batch (fp64 tables, differential rotation, more than comp::kMaxBins mu bins, several devices): per-star launches
    // dealt to three lanes
    cudaStream_t lanes[3];
    int rc = batch_fork(s0, st, lanes);
    if (rc) return rc;
    int first_error = SOAP_OK;
    for (int k = 0; k < n_stars && !first_error; ++k) first_error = soap_integrate_quiet(stars[k], quiet[k], out[k], lanes[k % 3]);
    rc = batch_join(s0, st, lanes);  // joined even after an error: no dangling lane
    return first_error ? first_error : rc;
}

int soap_batch_active_timeseries(soap_star *const *stars, int32_t n_stars, const soap_spectra *const *quiet,
                                 const soap_spectra *const *spot, const soap_spectra *const *facula,
                                 const soap_region *const *regions, const int32_t *n_regions, const double *const *phases,
                                 const int32_t *n_phases, void *const *out_delta, const int64_t *out_pitch, void *stream) {
    if (!stars || !quiet || !regions || !n_regions || !phases || !n_phases || !out_delta || !out_pitch || n_stars < 0)
        return SOAP_ERR_INVALID_ARG;
    for (int k = 0; k < n_stars; ++k)
        if (!stars[k]) return SOAP_ERR_INVALID_ARG;
    if (n_stars == 0) return SOAP_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    soap_star *s0 = stars[0];
    // ---- every argument of every star is checked before anything is enqueued ----------------------------------------
    bool one_launch = true;
    std::vector<ActiveCall> calls;
    calls.reserve((size_t)n_stars);
    for (int k = 0; k < n_stars; ++k) {
        soap_star *s = stars[k];
        const soap_spectra *sp = spot ? spot[k] : nullptr, *fa = facula ? facula[k] : nullptr;
        if (!s->ready) return s->fail(SOAP_ERR_NOT_READY, "soap_disk_geometry has not been called (star %d of the batch)", k);
        int rc = check_spectra(s, quiet[k], "quiet");
        if (rc) return rc;
        if (sp && ((rc = check_spectra(s, sp, "spot")) || (rc = check_same_grid(s, quiet[k], sp, "spot")))) return rc;
        if (fa && ((rc = check_spectra(s, fa, "facula")) || (rc = check_same_grid(s, quiet[k], fa, "facula")))) return rc;
        if ((rc = check_regions(s, regions[k], n_regions[k], phases[k], n_phases[k], sp, fa))) return rc;
        if (n_phases[k] > 0 && !out_delta[k]) return s->fail(SOAP_ERR_INVALID_ARG, "out_delta is NULL (star %d of the batch)", k);
        if (out_pitch[k] < quiet[k]->n_pix) return s->fail(SOAP_ERR_INVALID_ARG, "out_pitch must be >= n_pix (star %d of the batch)", k);
        for (int j = 0; j < k; ++j)
            if (stars[j] == s) return s->fail(SOAP_ERR_INVALID_ARG, "star %d appears twice in the batch", k);
        one_launch = one_launch && s->device == s0->device && quiet[k]->dtype == SOAP_F32 && s->prm.diff_rot == 0.0 &&
                     (s->form_used == SOAP_FORM_FIR) == (s0->form_used == SOAP_FORM_FIR);
        if (n_phases[k] > 0)
            calls.push_back(ActiveCall{s, quiet[k], sp, fa, regions[k], n_regions[k], phases[k], n_phases[k], nullptr, out_delta[k], out_pitch[k]});
    }
    if (calls.empty()) return SOAP_OK;
    SOAP_CUDA(s0, cudaSetDevice(s0->device));
    if (one_launch) {
        // ONE active-map launch and ONE shift-interpolate-accumulate launch for the batch (groups of f32::kMaxBatchStars)
        for (size_t k0 = 0; k0 < calls.size(); k0 += f32::kMaxBatchStars) {
            const int n = (int)std::min<size_t>(f32::kMaxBatchStars, calls.size() - k0);
            int rc = active_f32_launch(calls.data() + k0, n, SOAP_EFFECT_TOTAL, true, false, st);
            if (rc) return rc;
        }
        return SOAP_OK;
    }
    // mixed batch (fp64 tables, differential rotation, several devices): per-star launches dealt to three lanes
    cudaStream_t lanes[3];
    int rc = batch_fork(s0, st, lanes);
    if (rc) return rc;
    int first_error = SOAP_OK;
    for (int k = 0; k < n_stars && !first_error; ++k)
        first_error = soap_active_timeseries(stars[k], quiet[k], spot ? spot[k] : nullptr, facula ? facula[k] : nullptr, regions[k],
                                             n_regions[k], phases[k], n_phases[k], out_delta[k], out_pitch[k], nullptr, lanes[k % 3]);
    rc = batch_join(s0, st, lanes);
    return first_error ? first_error : rc;
}

}  // extern "C"
