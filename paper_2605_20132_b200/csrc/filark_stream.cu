// filark_stream.cu -- C ABI (include/filark_stream.h) + host-side preparation + launches.
//
// Host work per create: validate, rewrite every SOS section as a conditioned 2-state system
// (design.hpp), build the float64 block-power / fix-up tables, round to fp32, upload, zero the
// carried state.  Host work per push: argument checks, the tail-tile table for this n_t
// (cached), ONE kernel launch on the caller's stream.  No synchronisation, no allocation.
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <algorithm>
#include <map>
#include <unordered_map>
#include <vector>

#include "../../include/filark_stream.h"
#include "../../include/filark_debug.h"
#include "design.hpp"
#include "filark_kernels.cuh"
#include "filark_kernels_tr.cuh"

using namespace filark;

// Sub-block lengths compiled as kernel variants; a push picks the cheapest for its n_t.
static const int kVariantL[] = {8, 16, 24};
constexpr int kNumVariants = 3;
constexpr int kMaxL = 24;                // r0 < kMaxL: the tail a push leaves is shorter than its L
constexpr int kMaxDevices = 64;          // devices whose kernel attributes are tracked

struct filark_stream {
    int device;
    int n_ch, n_sec, sta_len, lta_len, layout;
    unsigned flags;
    Section sec[kMaxSec];
    bool lean_kinds;                // every section is kKindDF2 or kKindDelta: the smaller kernel serves
    double gain;
    void* proto[kNumVariants];      // host PushParams<L> with every table filled; pointers patched per push
    SerialParams serial;            // the same for the serial diagnostic kernel
    float* d_state;
    size_t state_floats;
    float* d_hist;                  // raw tail of the previous push: [n_ch][kHist] (both layouts)
    // trigger on the characteristic function (filark_stream_set_trigger): off while thr_on <= 0
    float thr_on, thr_off;
    Event* d_events;
    unsigned* d_n_events;
    unsigned ev_cap;
    CmCtl* d_cctl;                  // channel-major kernel: double-buffered control slots (filark_kernels.cuh)
    unsigned* d_progress;           // [n_ch] segments completed per channel (cumulative)
    // what the previous channel-major push touched: a push may overlap the one before it on the
    // device only if it follows it directly in the same stream and their buffers are disjoint
    int prev_valid;                 // how many of the entries below describe pushes that may still run
    cudaStream_t prev_stream;
    uintptr_t prev_lo[kCmDepth - 1][3], prev_hi[kCmDepth - 1][3];     // [0] = the push before, [1] = the one before that
    // zero-phase window mode (filark_stream_zero_phase): a second stream of the same cascade and two
    // window-sized temporaries, made on first use; the cascade as it was given
    double sos[6 * kMaxSec];
    filark_stream* zp;
    float* d_zp_tmp[2];
    size_t zp_elems;
    int n_sm;
    size_t smem_optin;
    int last_cuda_error;
    long long launches, samples;
    // staging for push_host: two sets of (in, filt, cf) used alternately, an upload and a download
    // stream of the handle's own, and the events that order them against the caller's stream
    float* d_stage[2][3];
    size_t stage_elems;
    cudaStream_t s_h2d, s_d2h;
    cudaEvent_t ev_h2d[2], ev_kernel[2], ev_d2h[2];
    bool host_ready, ev_pending[2];
    unsigned host_pushes;
};

// Last handle that launched on a stream (process-wide): a push that follows ANOTHER handle's push
// in the same stream must not start early either (its input may be that push's output).
static std::mutex g_reg_mutex;
static std::unordered_map<cudaStream_t, const filark_stream*> g_last_on_stream;

static bool registry_is_last(cudaStream_t s, const filark_stream* h)
{
    std::lock_guard<std::mutex> lock(g_reg_mutex);
    auto it = g_last_on_stream.find(s);
    return it != g_last_on_stream.end() && it->second == h;
}
static void registry_set(cudaStream_t s, const filark_stream* h)
{
    std::lock_guard<std::mutex> lock(g_reg_mutex);
    g_last_on_stream[s] = h;
}
static void registry_forget(const filark_stream* h)
{
    std::lock_guard<std::mutex> lock(g_reg_mutex);
    for (auto it = g_last_on_stream.begin(); it != g_last_on_stream.end();)
        it = it->second == h ? g_last_on_stream.erase(it) : ++it;
}

// Tuning switches: experiments only, compiled in with -DFK_TUNE (never in the product library,
// which reads no environment variable).
struct Tune { int warps; bool nopdl, small_ctas, all_kinds; };
static const Tune& tune()
{
#ifdef FK_TUNE
    static const Tune t = [] {
        Tune v{};
        const char* w = std::getenv("FILARK_TUNE_WARPS");
        v.warps = w ? std::atoi(w) : 0;
        v.nopdl = std::getenv("FILARK_TUNE_NOPDL") != nullptr;
        v.small_ctas = std::getenv("FILARK_TUNE_SMALL_CTAS") != nullptr;
        v.all_kinds = std::getenv("FILARK_TUNE_ALL_KINDS") != nullptr;
        return v;
    }();
#else
    static const Tune t{};
#endif
    return t;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute of a kernel: set it once
// per (kernel instance, device).  `done` is one word per template instance; bit d = device d.
static cudaError_t set_smem_attr_once(std::atomic<unsigned long long>& done, int device, const void* func, size_t bytes)
{
    const bool tracked = device >= 0 && device < kMaxDevices;
    if (tracked && ((done.load(std::memory_order_acquire) >> device) & 1ull)) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess && tracked) done.fetch_or(1ull << device, std::memory_order_release);
    return e;
}

static filark_status_t cuda_fail(filark_stream* h, cudaError_t e)
{
    if (h) h->last_cuda_error = (int)e;
    return FILARK_ERR_CUDA;
}

static void put_mat(float* dst, const Mat2& m)
{
    dst[0] = (float)m.a; dst[1] = (float)m.b; dst[2] = (float)m.c; dst[3] = (float)m.d;
}

// Everything of a push that does not depend on its buffers: tables in float64, rounded last.
template <int L> static void build_proto(const filark_stream* h, PushParams<L>* p)
{
    std::memset(p, 0, sizeof(*p));
    p->n_ch = h->n_ch; p->n_sec = h->n_sec; p->lta_len = h->lta_len;
    p->gain = (float)h->gain;
    p->ratio = (float)((double)h->lta_len / (double)h->sta_len);
    p->lta_thr = (float)(1e-30 * (double)h->lta_len);      // lta <= 1e-30  <=>  lta~ <= 1e-30 N_l
    for (int k = 0; k < h->n_sec; ++k) {
        const Section& s = h->sec[k];
        SecParams<L>& T = p->sec[k];
        T.kind = s.kind;
        for (int i = 0; i < 5; ++i) T.c[i] = (float)s.coef[i];
        put_mat(T.P, mpow(s.A, L));
        Mat2 q = mpow(s.A, 2 * L);
        int nsteps = kSteps;
        for (int d = 0; d < kSteps; ++d) {
            put_mat(T.Q[d], q);
            if (nsteps == kSteps && norm1(q) < 1e-10) nsteps = d;      // this and later steps add < 1e-10
            q = mul(q, q);
        }
        T.nsteps = nsteps;
        double g[2 * L];
        fixup_rows(s, L, g);
        for (int i = 0; i < L; ++i) { T.g[i][0] = (float)g[2 * i]; T.g[i][1] = (float)g[2 * i + 1]; }
    }
    const double cs = 1.0 / h->sta_len, cl = 1.0 / h->lta_len;
    AvgParams& a = p->avg;
    a.alpha[0] = (float)(1.0 - cs); a.alpha[1] = (float)(1.0 - cl);
    a.betaL[0] = (float)one_minus_pow(cs, L); a.betaL[1] = (float)one_minus_pow(cl, L);
    for (int d = 0; d < kSteps; ++d) {
        const double e = 2.0 * L * (double)(1 << d);
        a.betaQ[d][0] = (float)one_minus_pow(cs, e);
        a.betaQ[d][1] = (float)one_minus_pow(cl, e);
    }
    a.invN[0] = (float)cs; a.invN[1] = (float)cl;
}

static void build_serial(const filark_stream* h, SerialParams* p)
{
    std::memset(p, 0, sizeof(*p));
    p->n_ch = h->n_ch; p->n_sec = h->n_sec; p->lta_len = h->lta_len;
    p->gain = (float)h->gain;
    p->ratio = (float)((double)h->lta_len / (double)h->sta_len);
    p->lta_thr = (float)(1e-30 * (double)h->lta_len);
    p->inv_ns = (float)(1.0 / h->sta_len); p->inv_nl = (float)(1.0 / h->lta_len);
    for (int k = 0; k < h->n_sec; ++k) {
        p->kind[k] = h->sec[k].kind;
        for (int i = 0; i < 5; ++i) p->c[k][i] = (float)h->sec[k].coef[i];
    }
}

static void* alloc_proto(int v, const filark_stream* h)
{
    switch (kVariantL[v]) {
#define FK_CASE(LL) case LL: { auto* p = (PushParams<LL>*)std::malloc(sizeof(PushParams<LL>)); if (p) build_proto<LL>(h, p); return p; }
        FK_CASE(8) FK_CASE(16)
        default: { auto* p = (PushParams<24>*)std::malloc(sizeof(PushParams<24>)); if (p) build_proto<24>(h, p); return p; }
#undef FK_CASE
    }
}

// Variant for a push of n_t samples.  Measured on B200 (profiles/): L = 24 with 16 warps per SM
// is the fastest per sample (larger L costs warps, smaller L more scans per sample), so it is
// used unless a smaller L puts a short push into fewer lane-samples: the cost of a tile is its
// L samples per lane-half plus a fixed part (scans, staging).  r0 is not known on the host
// and is taken as 0.
static int choose_variant(long long n_t)
{
    int best = 0; double best_cost = 1e300;
    for (int v = 0; v < kNumVariants; ++v) {
        const int L = kVariantL[v];
        const long long slots = (n_t + L - 1) / L;
        const double cost = (double)((slots + 63) / 64) * (L + 10.0);
        if (cost < best_cost * (1.0 - 1e-9) || (cost <= best_cost * (1.0 + 1e-9) && L == 24)) { best_cost = cost; best = v; }
    }
    return best;
}

static Geom geometry_rt(int L, unsigned r0, int n_t, bool vec4)
{
    switch (L) {
        case 8: return make_geom<8>(r0, n_t, vec4);
        case 16: return make_geom<16>(r0, n_t, vec4);
        default: return make_geom<24>(r0, n_t, vec4);
    }
}

// CTAS CTAs per SM, W warps per CTA; fewer warps per CTA, on more SMs, when there are few
// channels.  Every CTA of a push fits on the device at once (the segment waits rely on it).
template <int L, int CTAS, int kForm, bool kDyn, bool kShift>
static cudaError_t launch_cm_shift(const PushParams<L>& p, int device, int grid, int W, size_t smem, size_t smem_max, cudaStream_t stream)
{
    static std::atomic<unsigned long long> attr_done{0};
    const cudaError_t e = set_smem_attr_once(attr_done, device, (const void*)filark_push_cm_kernel<L, CTAS, kForm, false, kDyn, kShift>, smem_max);
    if (e != cudaSuccess) return e;
    // programmatic stream serialization: the kernel lets its dependents launch as soon as it has read
    // its control slot, and orders itself against the previous push channel by channel
    // (filark_kernels.cuh); p.wait_prior = 1 makes it an ordinary dependent launch
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)(W * 32));
    cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = tune().nopdl ? 0 : 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, filark_push_cm_kernel<L, CTAS, kForm, false, kDyn, kShift>, p);
}

// Rows that are not 16-byte aligned (p.vec4 = 0: some pointer, pitch or chunk length is not a multiple of
// four floats): the build of the kernel with the unrolled shifted paths (L = 24 only; filark_kernels.cuh).
template <int L, int CTAS, int kForm, bool kDyn>
static cudaError_t launch_cm_variant(const PushParams<L>& p, int device, int grid, int W, size_t smem, size_t smem_max, cudaStream_t stream)
{
    if constexpr (L == 24) {
        if (!p.vec4) return launch_cm_shift<L, CTAS, kForm, kDyn, true>(p, device, grid, W, smem, smem_max, stream);
    }
    return launch_cm_shift<L, CTAS, kForm, kDyn, false>(p, device, grid, W, smem, smem_max, stream);
}

// Tiles per channel of a launch: the r0 = 0 estimate and the largest number whatever r0 < kMaxL the
// first chunk finds waiting (a later chunk's r0 follows from the first one's).
template <int L> static void launch_tiles(const PushParams<L>& p, long long* est, long long* most)
{
    long long e = 0, m = 0;
    for (int k = 0; k < p.n_push; ++k) {
        e += ((long long)p.ck[k].n_t + L - 1) / L / 64 + 1;
        m += (((long long)p.ck[k].n_t + kMaxL - 1 + L - 1) / L + 63) / 64;
    }
    *est = e; *most = m;
}

// Tiles per work item: about 8 items per warp of the grid.  (Not evened out: a short last segment
// per channel is welcome -- items are taken in rising order, so the short ones fill the end of the launch.)
static int segment_tiles(long long n_tiles, long long units, long long workers)
{
    const long long st = n_tiles * units / (8LL * workers);
    return (int)(st < 1 ? 1 : (st > 0x3fffffff ? 0x3fffffff : st));
}

template <int L, int CTAS, int kForm>
static cudaError_t launch_cm_shape(const filark_stream* h, PushParams<L>& p, cudaStream_t stream)
{
    const size_t warp_bytes = sizeof(float) * (size_t)warp_smem_floats<L>();
    int per_sm = cm_max_warps<L>();                      // warps per SM
    const int fit = (int)((h->smem_optin - 256) / warp_bytes);
    if (fit < per_sm) per_sm = fit;
    int W = cm_cta_warps<L, CTAS>();
    if (W > per_sm) W = per_sm;
    const int want = (p.n_ch + h->n_sm - 1) / h->n_sm;
    if (want < W) W = want;
    if (tune().warps >= 1 && tune().warps <= W) W = tune().warps;       // tuning experiments only
    if (W < 1) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)W * warp_bytes;
    int grid = (p.n_ch + W - 1) / W;
    const int resident = h->n_sm * (per_sm / W < 16 ? per_sm / W : 16);
    if (grid > resident) grid = resident;
    // work items: runs of seg_tiles tiles of a channel
    long long n_tiles, n_tiles_max;
    launch_tiles<L>(p, &n_tiles, &n_tiles_max);
    p.seg_tiles = segment_tiles(n_tiles, p.n_ch, (long long)grid * W);
    // one segment per channel for certain: static work distribution; otherwise items are claimed
    // (filark_kernels.cuh, "Work items").  Long pushes (CTAS = 1) always claim.
    const size_t smem_max = (size_t)cm_cta_warps<L, CTAS>() * warp_bytes;
    if constexpr (CTAS != 1) {
        if (p.seg_tiles >= n_tiles_max)
            return launch_cm_variant<L, CTAS, kForm, false>(p, h->device, grid, W, smem, smem_max, stream);
    }
    return launch_cm_variant<L, CTAS, kForm, true>(p, h->device, grid, W, smem, smem_max, stream);
}

// Kernel form (filark_kernels.cuh, process_tile): bit 0 = every section form (not only the two a Butterworth
// band-pass gives), bit 1 = the trigger.
static int kernel_form(const filark_stream* h) { return (h->thr_on > 0.0f ? 2 : 0) + (h->lean_kinds ? 0 : 1); }

// Launch shape (filark_kernels.cuh): one CTA per SM when every resident warp gets a long run of tiles
// anyway, small CTAs otherwise.  (L = 24 is the only variant long pushes ever use.)
template <int L>
static cudaError_t launch_cm(const filark_stream* h, PushParams<L>& p, cudaStream_t stream)
{
    const int form = kernel_form(h);
    if constexpr (L == 24 || (L == 16 && FK_MAXW16 != 16)) {
        long long n_tiles, n_tiles_max;
        launch_tiles<L>(p, &n_tiles, &n_tiles_max);
        const bool long_push = n_tiles_max * p.n_ch >= 12LL * h->n_sm * cm_max_warps<L>();
        if (long_push && !tune().small_ctas)
            return form == 0 ? launch_cm_shape<L, 1, 0>(h, p, stream)
                             : (form == 1 ? launch_cm_shape<L, 1, 1>(h, p, stream)
                                          : (form == 2 ? launch_cm_shape<L, 1, 2>(h, p, stream) : launch_cm_shape<L, 1, 3>(h, p, stream)));
    }
    return form == 0 ? launch_cm_shape<L, kCmCtasPerSm, 0>(h, p, stream)
                     : (form == 1 ? launch_cm_shape<L, kCmCtasPerSm, 1>(h, p, stream)
                                  : (form == 2 ? launch_cm_shape<L, kCmCtasPerSm, 2>(h, p, stream) : launch_cm_shape<L, kCmCtasPerSm, 3>(h, p, stream)));
}

// Time-major chunks: the same kernel with the transpose in shared memory (filark_kernels.cuh): one CTA
// of kTmChannels warps per SM, work items = (segment, group of kTmChannels adjacent channels).
template <int L, int kForm>
static cudaError_t launch_tm_kinds(const filark_stream* h, PushParams<L>& p, cudaStream_t stream)
{
    const size_t smem = sizeof(float) * (size_t)kTmChannels * (size_t)warp_stride<L, true>();
    const int n_cg = (p.n_ch + kTmChannels - 1) / kTmChannels;
    const int grid = n_cg < h->n_sm ? n_cg : h->n_sm;
    long long n_tiles, n_tiles_max;
    launch_tiles<L>(p, &n_tiles, &n_tiles_max);
    p.seg_tiles = segment_tiles(n_tiles, n_cg, grid);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)(kTmChannels * 32));
    cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = tune().nopdl ? 0 : 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (p.seg_tiles >= n_tiles_max) {
        static std::atomic<unsigned long long> attr_done{0};
        const cudaError_t e = set_smem_attr_once(attr_done, h->device, (const void*)filark_push_cm_kernel<L, 1, kForm, true, false>, smem);
        if (e != cudaSuccess) return e;
        return cudaLaunchKernelEx(&cfg, filark_push_cm_kernel<L, 1, kForm, true, false>, p);
    }
    static std::atomic<unsigned long long> attr_done{0};
    const cudaError_t e = set_smem_attr_once(attr_done, h->device, (const void*)filark_push_cm_kernel<L, 1, kForm, true, true>, smem);
    if (e != cudaSuccess) return e;
    return cudaLaunchKernelEx(&cfg, filark_push_cm_kernel<L, 1, kForm, true, true>, p);
}
template <int L>
static cudaError_t launch_tm(const filark_stream* h, PushParams<L>& p, cudaStream_t stream)
{
    const int form = kernel_form(h);
    return form == 0 ? launch_tm_kinds<L, 0>(h, p, stream)
                     : (form == 1 ? launch_tm_kinds<L, 1>(h, p, stream)
                                  : (form == 2 ? launch_tm_kinds<L, 2>(h, p, stream) : launch_tm_kinds<L, 3>(h, p, stream)));
}

// Time-major chunks with one channel per LANE (filark_kernels_tr.cuh): one CTA of 16 warps per SM, work items =
// (segment, block of 32 channels), always claimed.
template <int kForm>
static cudaError_t launch_tr_kinds(const filark_stream* h, PushParams<kTrL>& p, cudaStream_t stream)
{
    const int n_cb = (p.n_ch + kTrCh - 1) / kTrCh;
    const int grid = n_cb < h->n_sm ? n_cb : h->n_sm;
    long long n_tiles = 0;
    for (int k = 0; k < p.n_push; ++k) n_tiles += ((long long)p.ck[k].n_t + kTrL - 1) / kTrL / 32 + 1;
    p.seg_tiles = segment_tiles(n_tiles, n_cb, grid);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)(kTrWarps * 32));
    cfg.dynamicSmemBytes = kTrSmemBytes; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = tune().nopdl ? 0 : 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    static std::atomic<unsigned long long> attr_done{0};
    const cudaError_t e = set_smem_attr_once(attr_done, h->device, (const void*)filark_push_tr_kernel<kForm>, kTrSmemBytes);
    if (e != cudaSuccess) return e;
    return cudaLaunchKernelEx(&cfg, filark_push_tr_kernel<kForm>, p);
}
static cudaError_t launch_tr(const filark_stream* h, PushParams<kTrL>& p, cudaStream_t stream)
{
    return kernel_form(h) == 0 ? launch_tr_kinds<0>(h, p, stream) : launch_tr_kinds<1>(h, p, stream);
}

// One chunk as the caller describes it (all pushes end up here).
struct ChunkArgs {
    const float* in; long long n_t, in_pitch;
    float* filt; float* cf; long long out_pitch;
};

template <int L>
static cudaError_t push_variant(const filark_stream* h, int v, const ChunkArgs* c, int n, int vec4, int wait_prior,
                                cudaStream_t stream, bool lanes = false)
{
    PushParams<L> p = *(const PushParams<L>*)h->proto[v];
    p.state = h->d_state; p.hist = h->d_hist; p.cctl = h->d_cctl; p.progress = h->d_progress;
    p.n_push = n; p.vec4 = vec4; p.wait_prior = wait_prior;
    p.thr_on = h->thr_on; p.thr_off = h->thr_off; p.events = h->d_events; p.n_events = h->d_n_events; p.ev_cap = h->ev_cap;
    unsigned t_cum = 0;
    for (int k = 0; k < n; ++k) {
        Chunk& d = p.ck[k];
        d.in = c[k].in; d.filt = c[k].filt; d.cf = c[k].cf;
        d.in_pitch = c[k].in_pitch; d.out_pitch = c[k].out_pitch;
        d.n_t = (int)c[k].n_t; d.n_base = (int)(c[k].n_t / L); d.n_rem = (int)(c[k].n_t % L);
        d.t_cum = t_cum;
        t_cum += (unsigned)c[k].n_t;
    }
    if constexpr (L == kTrL) {
        if (lanes) return launch_tr(h, p, stream);
    }
    if (h->layout == FILARK_LAYOUT_TIME_MAJOR) return launch_tm<L>(h, p, stream);
    return launch_cm<L>(h, p, stream);
}

extern "C" {

const char* filark_status_string(filark_status_t s)
{
    switch (s) {
        case FILARK_OK: return "ok";
        case FILARK_ERR_INVALID_ARG: return "invalid argument";
        case FILARK_ERR_UNSTABLE: return "unstable section (pole radius >= 1)";
        case FILARK_ERR_ALLOC: return "allocation failed";
        case FILARK_ERR_CUDA: return "CUDA error";
        case FILARK_ERR_DEVICE_MISMATCH: return "current device differs from the handle's device";
        case FILARK_ERR_ALIGNMENT: return "device pointer not 4-byte aligned";
        case FILARK_ERR_TOO_LARGE: return "more channels than the fixed device scratch of filark_stream_once_noalloc holds";
    }
    return "unknown status";
}

int filark_last_cuda_error(const filark_stream_t* h) { return h ? h->last_cuda_error : 0; }
long long filark_stream_launch_count(const filark_stream_t* h) { return h ? h->launches : -1; }
long long filark_stream_samples_pushed(const filark_stream_t* h) { return h ? h->samples : -1; }

static filark_status_t design_all(const double* sos, int n_sec, Section* sec, double* gain)
{
    double g = 1.0;
    for (int k = 0; k < n_sec; ++k) {
        const DesignStatus ds = design_section(sos + 6 * k, &sec[k]);
        if (ds == DESIGN_INVALID) return FILARK_ERR_INVALID_ARG;
        if (ds == DESIGN_UNSTABLE) return FILARK_ERR_UNSTABLE;
        g *= sec[k].gain;
    }
    if (!std::isfinite(g)) return FILARK_ERR_INVALID_ARG;
    *gain = g;
    return FILARK_OK;
}

static filark_status_t check_create_args(const void* out, int n_ch, const double* sos, int n_sec,
                                         int sta_len, int lta_len, int layout, unsigned flags)
{
    if (!out || !sos || n_ch <= 0 || n_sec <= 0 || n_sec > FILARK_MAX_SECTIONS) return FILARK_ERR_INVALID_ARG;
    if (sta_len < 1 || lta_len < sta_len) return FILARK_ERR_INVALID_ARG;
    if (layout != FILARK_LAYOUT_CHANNEL_MAJOR && layout != FILARK_LAYOUT_TIME_MAJOR) return FILARK_ERR_INVALID_ARG;
    if (flags & ~(FILARK_FLAG_SERIAL_SCAN | FILARK_FLAG_STRICT_ORDER | FILARK_FLAG_OVERLAP_PUSHES | FILARK_FLAG_TM_TRANSPOSE | 0xFF00u)) return FILARK_ERR_INVALID_ARG;
    if (flags & 0xFF00u) {
        bool ok = false;
        for (int v = 0; v < kNumVariants; ++v) ok = ok || kVariantL[v] == (int)((flags >> 8) & 0xFF);
        if (!ok) return FILARK_ERR_INVALID_ARG;
    }
    return FILARK_OK;
}

filark_status_t filark_stream_create_ex(filark_stream_t** out, int n_ch, const double* sos, int n_sec,
                                        int sta_len, int lta_len, int layout, unsigned flags)
{
    filark_status_t st = check_create_args(out, n_ch, sos, n_sec, sta_len, lta_len, layout, flags);
    if (st != FILARK_OK) return st;
    filark_stream* h = new (std::nothrow) filark_stream();
    if (!h) return FILARK_ERR_ALLOC;
    std::memset(h, 0, sizeof(*h));
    st = design_all(sos, n_sec, h->sec, &h->gain);
    if (st != FILARK_OK) { delete h; return st; }
    h->lean_kinds = !tune().all_kinds;
    for (int k = 0; k < n_sec; ++k) h->lean_kinds = h->lean_kinds && (h->sec[k].kind == kKindDF2 || h->sec[k].kind == kKindDelta);
    h->n_ch = n_ch; h->n_sec = n_sec; h->sta_len = sta_len; h->lta_len = lta_len;
    h->layout = layout; h->flags = flags;
    std::memcpy(h->sos, sos, sizeof(double) * 6 * (size_t)n_sec);
    h->state_floats = (size_t)n_ch * (size_t)state_floats(n_sec);
    cudaError_t e = cudaGetDevice(&h->device);
    int optin = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    h->smem_optin = (size_t)optin;
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_state, sizeof(float) * h->state_floats);
    if (e == cudaSuccess) e = cudaMemset(h->d_state, 0, sizeof(float) * h->state_floats);
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_hist, sizeof(float) * (size_t)n_ch * kHist);
    if (e == cudaSuccess) e = cudaMemset(h->d_hist, 0, sizeof(float) * (size_t)n_ch * kHist);
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_cctl, sizeof(CmCtl));
    if (e == cudaSuccess) e = cudaMemset(h->d_cctl, 0, sizeof(CmCtl));
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_progress, sizeof(unsigned) * (size_t)n_ch);
    if (e == cudaSuccess) e = cudaMemset(h->d_progress, 0, sizeof(unsigned) * (size_t)n_ch);
    bool host_oom = false;
    build_serial(h, &h->serial);
    for (int v = 0; v < kNumVariants && e == cudaSuccess && !host_oom; ++v) {
        h->proto[v] = alloc_proto(v, h);
        if (!h->proto[v]) host_oom = true;
    }
    if (e != cudaSuccess || host_oom) {
        const bool oom = host_oom || e == cudaErrorMemoryAllocation;
        for (int v = 0; v < kNumVariants; ++v) std::free(h->proto[v]);
        cudaFree(h->d_state); cudaFree(h->d_hist); cudaFree(h->d_cctl); cudaFree(h->d_progress);
        delete h;
        cudaGetLastError();
        return oom ? FILARK_ERR_ALLOC : FILARK_ERR_CUDA;
    }
    *out = h;
    return FILARK_OK;
}

filark_status_t filark_stream_create(filark_stream_t** out, int n_ch, const double* sos, int n_sec,
                                     int sta_len, int lta_len)
{
    return filark_stream_create_ex(out, n_ch, sos, n_sec, sta_len, lta_len,
                                   FILARK_LAYOUT_CHANNEL_MAJOR, FILARK_FLAG_NONE);
}

filark_status_t filark_stream_destroy(filark_stream_t* h)
{
    if (!h) return FILARK_OK;
    registry_forget(h);
    // everything the handle owns lives on h->device, whatever device is current now
    int cur = -1;
    const bool have_cur = cudaGetDevice(&cur) == cudaSuccess;
    const bool switched = have_cur && cur != h->device && cudaSetDevice(h->device) == cudaSuccess;
    cudaDeviceSynchronize();
    for (int v = 0; v < kNumVariants; ++v) std::free(h->proto[v]);
    cudaFree(h->d_state); cudaFree(h->d_hist); cudaFree(h->d_cctl); cudaFree(h->d_progress);
    cudaFree(h->d_events); cudaFree(h->d_n_events);
    cudaFree(h->d_zp_tmp[0]); cudaFree(h->d_zp_tmp[1]);
    if (h->zp) { filark_stream* z = h->zp; h->zp = nullptr; filark_stream_destroy(z); }
    for (int j = 0; j < 2; ++j) for (int i = 0; i < 3; ++i) cudaFree(h->d_stage[j][i]);
    if (h->host_ready) {
        cudaStreamDestroy(h->s_h2d); cudaStreamDestroy(h->s_d2h);
        for (int j = 0; j < 2; ++j) { cudaEventDestroy(h->ev_h2d[j]); cudaEventDestroy(h->ev_kernel[j]); cudaEventDestroy(h->ev_d2h[j]); }
    }
    if (switched) cudaSetDevice(cur);
    cudaGetLastError();
    delete h;
    return FILARK_OK;
}

filark_status_t filark_stream_reset(filark_stream_t* h, cudaStream_t stream)
{
    if (!h) return FILARK_ERR_INVALID_ARG;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(h, e);
    if (dev != h->device) return FILARK_ERR_DEVICE_MISMATCH;
    e = cudaMemsetAsync(h->d_state, 0, sizeof(float) * h->state_floats, stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->d_cctl, 0, sizeof(CmCtl), stream);
    h->prev_valid = 0;
    if (e == cudaSuccess) e = cudaMemsetAsync(h->d_progress, 0, sizeof(unsigned) * (size_t)h->n_ch, stream);
    if (e != cudaSuccess) return cuda_fail(h, e);
    h->samples = 0;
    return FILARK_OK;
}

static bool overlaps(const void* a, size_t na, const void* b, size_t nb)
{
    const uintptr_t a0 = (uintptr_t)a, b0 = (uintptr_t)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

// Argument checks of one chunk (include/filark_stream.h, filark_stream_push); the byte extents of its buffers.
static filark_status_t check_chunk(const filark_stream* h, const ChunkArgs& c, size_t* in_bytes, size_t* out_bytes)
{
    if (c.n_t < 1 || c.n_t > 0x7fff0000LL) return FILARK_ERR_INVALID_ARG;     // samples per channel of one chunk fit an int
    if (!c.in || (!c.filt && !c.cf)) return FILARK_ERR_INVALID_ARG;
    const bool cm = h->layout == FILARK_LAYOUT_CHANNEL_MAJOR;
    const long long row_len = cm ? c.n_t : (long long)h->n_ch;
    const long long n_rows = cm ? (long long)h->n_ch : c.n_t;
    if (c.in_pitch < row_len || c.out_pitch < row_len) return FILARK_ERR_INVALID_ARG;
    if (((uintptr_t)c.in | (uintptr_t)c.filt | (uintptr_t)c.cf) & 3u) return FILARK_ERR_ALIGNMENT;
    *in_bytes = sizeof(float) * (size_t)((n_rows - 1) * c.in_pitch + row_len);
    *out_bytes = sizeof(float) * (size_t)((n_rows - 1) * c.out_pitch + row_len);
    if ((c.filt && overlaps(c.in, *in_bytes, c.filt, *out_bytes)) ||
        (c.cf && overlaps(c.in, *in_bytes, c.cf, *out_bytes)) ||
        (c.filt && c.cf && overlaps(c.filt, *out_bytes, c.cf, *out_bytes)))
        return FILARK_ERR_INVALID_ARG;
    return FILARK_OK;
}

// Sub-block length for a launch: the cheapest variant over its chunks (every chunk has tiles of its own).
static int choose_variant_chunks(const filark_stream* h, const ChunkArgs* c, int n)
{
    for (int i = 0; i < kNumVariants; ++i) if (kVariantL[i] == (int)((h->flags >> 8) & 0xFF)) return i;
    if (n == 1) return choose_variant(c[0].n_t);
    int best = kNumVariants - 1; double best_cost = 1e300;
    for (int v = 0; v < kNumVariants; ++v) {
        const int L = kVariantL[v];
        double cost = 0.0;
        for (int k = 0; k < n; ++k) cost += (double)(((c[k].n_t + L - 1) / L + 63) / 64) * (L + 10.0);
        if (cost < best_cost * (1.0 - 1e-9) || (cost <= best_cost * (1.0 + 1e-9) && L == 24)) { best_cost = cost; best = v; }
    }
    return best;
}

// ONE launch over n <= kMaxBatch checked chunks (consecutive in the stream of samples).  may_overlap:
// the caller knows that nothing but this handle's own previous launch lies between that launch and
// this one in `stream` (filark_stream.h, "Ordering").
static filark_status_t launch_chunks(filark_stream_t* h, const ChunkArgs* c, int n, cudaStream_t stream, bool may_overlap)
{
    const bool cm = h->layout == FILARK_LAYOUT_CHANNEL_MAJOR;
    cudaError_t e = cudaSuccess;
    long long total = 0;
    for (int k = 0; k < n; ++k) total += c[k].n_t;
    if (h->flags & FILARK_FLAG_SERIAL_SCAN) {
        // Serial diagnostic kernel (either layout), chunk by chunk.
        const int ns = state_floats(h->n_sec);
        for (int k = 0; k < n && e == cudaSuccess; ++k) {
            SerialParams p = h->serial;
            p.in = c[k].in; p.filt = c[k].filt; p.cf = c[k].cf; p.state = h->d_state; p.n_t = c[k].n_t;
            p.sc_in = cm ? c[k].in_pitch : 1; p.st_in = cm ? 1 : c[k].in_pitch;
            p.sc_out = cm ? c[k].out_pitch : 1; p.st_out = cm ? 1 : c[k].out_pitch;
            p.state_sc = cm ? ns : 1; p.state_sk = cm ? 1 : h->n_ch;
            const int block = 128, grid = (h->n_ch + block - 1) / block;
            filark_push_serial_kernel<<<grid, block, 0, stream>>>(p);
            e = cudaGetLastError();
            if (e == cudaSuccess) h->launches += 1;
        }
    } else {
        int v = choose_variant_chunks(h, c, n);
        // time-major: the kernel with one channel per lane (filark_kernels_tr.cuh) unless a trigger is set, another
        // sub-block length is forced, or a pitch is too long for its 32-bit row offsets
        const unsigned force_L = (h->flags >> 8) & 0xFFu;
        bool lanes = !cm && kernel_form(h) < 2 && !(h->flags & FILARK_FLAG_TM_TRANSPOSE) && (force_L == 0 || force_L == (unsigned)kTrL);
        for (int k = 0; k < n && lanes; ++k) lanes = c[k].in_pitch < (1LL << 25) && c[k].out_pitch < (1LL << 25);
        // (a launch of fewer than four of its tiles per channel is over before its warps have fallen into step:
        // measured on separate 1,500-sample pushes, 171 against 190 Gsample/s for the transposing kernel)
        if (total < 4LL * kTrRows) lanes = false;
        if (lanes) for (int i = 0; i < kNumVariants; ++i) if (kVariantL[i] == kTrL) v = i;
        // bounding ranges of what the launch reads ([0]) and writes ([1] filt, [2] cf); alignment
        uintptr_t lo[3] = {~(uintptr_t)0, ~(uintptr_t)0, ~(uintptr_t)0}, hi[3] = {0, 0, 0};
        int vec4 = 1;
        for (int k = 0; k < n; ++k) {
            size_t ib = 0, ob = 0;
            check_chunk(h, c[k], &ib, &ob);
            const uintptr_t l3[3] = {(uintptr_t)c[k].in, (uintptr_t)c[k].filt, (uintptr_t)c[k].cf};
            const size_t b3[3] = {ib, ob, ob};
            for (int i = 0; i < 3; ++i)
                if (l3[i]) { if (l3[i] < lo[i]) lo[i] = l3[i]; if (l3[i] + b3[i] > hi[i]) hi[i] = l3[i] + b3[i]; }
            const uintptr_t all = l3[0] | l3[1] | l3[2];
            // (channel-major: introspection only; time-major: output rows allow 16-byte stores)
            const bool ok = cm ? ((all & 15u) == 0 && (c[k].in_pitch & 3) == 0 && (c[k].out_pitch & 3) == 0 && (c[k].n_t & 3) == 0)
                               : (((l3[1] | l3[2]) & 15u) == 0 && (c[k].out_pitch & 3) == 0);
            if (!ok) vec4 = 0;
        }
        // May this launch overlap the one before it?  Only if that was this handle's own launch, directly
        // before it in the same stream as far as this library launched anything, and the two share no
        // buffer (bounding ranges; filark_stream.h, "Ordering").
        int wait_prior = 1;
        if (may_overlap && !(h->flags & FILARK_FLAG_STRICT_ORDER) && h->prev_valid > 0 && h->prev_stream == stream &&
            registry_is_last(stream, h)) {
            bool clash = false;
            for (int q = 0; q < h->prev_valid; ++q)
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j)
                        if ((i > 0 || j > 0) && hi[i] && h->prev_hi[q][j] && lo[i] < h->prev_hi[q][j] &&
                            h->prev_lo[q][j] < hi[i])
                            clash = true;
            wait_prior = clash ? 1 : 0;
        }
        const int n_prev = wait_prior ? 0 : h->prev_valid;       // a waiting launch leaves nothing in flight behind it
        h->prev_valid = 0;
        switch (kVariantL[v]) {
            case 8: e = push_variant<8>(h, v, c, n, vec4, wait_prior, stream); break;
            case 16: e = push_variant<16>(h, v, c, n, vec4, wait_prior, stream); break;
            default: e = push_variant<24>(h, v, c, n, vec4, wait_prior, stream, lanes); break;
        }
        if (e == cudaSuccess) {
            const int keep = n_prev < kCmDepth - 2 ? n_prev : kCmDepth - 2;
            for (int q = keep; q > 0; --q)
                for (int i = 0; i < 3; ++i) { h->prev_lo[q][i] = h->prev_lo[q - 1][i]; h->prev_hi[q][i] = h->prev_hi[q - 1][i]; }
            for (int i = 0; i < 3; ++i) { h->prev_lo[0][i] = hi[i] ? lo[i] : 0; h->prev_hi[0][i] = hi[i]; }
            h->prev_valid = keep + 1; h->prev_stream = stream;
            h->launches += 1;
        }
    }
    registry_set(stream, h);
    if (e != cudaSuccess) return cuda_fail(h, e);
    h->samples += total;
    return FILARK_OK;
}

static filark_status_t check_device(filark_stream_t* h)
{
    int dev = -1;
    const cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(h, e);
    return dev != h->device ? FILARK_ERR_DEVICE_MISMATCH : FILARK_OK;
}

// One push = one launch over one chunk.
static filark_status_t push_impl(filark_stream_t* h, const float* d_in, long long n_t,
                                 long long in_pitch, float* d_filt, float* d_cf,
                                 long long out_pitch, cudaStream_t stream, bool may_overlap)
{
    if (!h || n_t < 0) return FILARK_ERR_INVALID_ARG;
    if (n_t == 0) return FILARK_OK;
    const ChunkArgs c{d_in, n_t, in_pitch, d_filt, d_cf, out_pitch};
    size_t ib = 0, ob = 0;
    filark_status_t st = check_chunk(h, c, &ib, &ob);
    if (st == FILARK_OK) st = check_device(h);
    if (st != FILARK_OK) return st;
    return launch_chunks(h, &c, 1, stream, may_overlap);
}

filark_status_t filark_stream_push_pitched(filark_stream_t* h, const float* d_in, long long n_t,
                                           long long in_pitch, float* d_filt, float* d_cf,
                                           long long out_pitch, cudaStream_t stream)
{
    if (!h) return FILARK_ERR_INVALID_ARG;
    return push_impl(h, d_in, n_t, in_pitch, d_filt, d_cf, out_pitch, stream, (h->flags & FILARK_FLAG_OVERLAP_PUSHES) != 0);
}

filark_status_t filark_stream_push(filark_stream_t* h, const float* d_in, long long n_t,
                                   float* d_filt, float* d_cf, cudaStream_t stream)
{
    if (!h) return FILARK_ERR_INVALID_ARG;
    const long long pitch = h->layout == FILARK_LAYOUT_CHANNEL_MAJOR ? n_t : (long long)h->n_ch;
    return push_impl(h, d_in, n_t, pitch, d_filt, d_cf, pitch, stream, (h->flags & FILARK_FLAG_OVERLAP_PUSHES) != 0);
}

// Does any buffer written by one chunk of the schedule overlap a buffer of ANOTHER chunk?  (Then the
// chunks cannot share a launch: inside a launch a channel's next tile is requested before the
// outputs of the tile before it are stored.)  Sweep over the ranges sorted by start address.
static bool schedule_aliases(const filark_stream* h, const ChunkArgs* c, int n)
{
    struct R { uintptr_t lo, hi; int out; };
    std::vector<R> r;
    r.reserve(3 * (size_t)n);
    for (int k = 0; k < n; ++k) {
        size_t ib = 0, ob = 0;
        check_chunk(h, c[k], &ib, &ob);
        r.push_back({(uintptr_t)c[k].in, (uintptr_t)c[k].in + ib, 0});
        if (c[k].filt) r.push_back({(uintptr_t)c[k].filt, (uintptr_t)c[k].filt + ob, 1});
        if (c[k].cf) r.push_back({(uintptr_t)c[k].cf, (uintptr_t)c[k].cf + ob, 1});
    }
    std::sort(r.begin(), r.end(), [](const R& a, const R& b) { return a.lo < b.lo; });
    uintptr_t end_any = 0, end_out = 0;            // furthest end of the ranges seen so far: all / written ones
    for (const R& x : r) {
        if (x.out ? x.lo < end_any : x.lo < end_out) return true;
        if (x.hi > end_any) end_any = x.hi;
        if (x.out && x.hi > end_out) end_out = x.hi;
    }
    return false;
}

filark_status_t filark_stream_push_many(filark_stream_t* h, int n_push, const float* const* d_in,
                                        const long long* n_t, float* const* d_filt, float* const* d_cf,
                                        cudaStream_t stream)
{
    if (!h || n_push < 0 || (n_push > 0 && (!d_in || !n_t))) return FILARK_ERR_INVALID_ARG;
    // the whole schedule is checked before anything is enqueued
    std::vector<ChunkArgs> c;
    c.reserve((size_t)n_push);
    for (int i = 0; i < n_push; ++i) {
        if (n_t[i] < 0) return FILARK_ERR_INVALID_ARG;
        if (n_t[i] == 0) continue;
        const long long pitch = h->layout == FILARK_LAYOUT_CHANNEL_MAJOR ? n_t[i] : (long long)h->n_ch;
        const ChunkArgs a{d_in[i], n_t[i], pitch, d_filt ? d_filt[i] : nullptr, d_cf ? d_cf[i] : nullptr, pitch};
        size_t ib = 0, ob = 0;
        const filark_status_t st = check_chunk(h, a, &ib, &ob);
        if (st != FILARK_OK) return st;
        c.push_back(a);
    }
    if (c.empty()) return FILARK_OK;
    const filark_status_t sd = check_device(h);
    if (sd != FILARK_OK) return sd;
    // Chunks that share no buffer go into common launches of up to kMaxBatch chunks (and < 2^31 samples
    // per channel): the carried state then never leaves the SM between them.  Otherwise, and with
    // FILARK_FLAG_STRICT_ORDER, one launch per chunk.
    const int n = (int)c.size();
    const bool fuse = !(h->flags & (FILARK_FLAG_STRICT_ORDER | FILARK_FLAG_SERIAL_SCAN)) && n > 1 && !schedule_aliases(h, c.data(), n);
    bool first = true;
    for (int i = 0; i < n;) {
        int m = 1;
        if (fuse) {
            long long tot = c[i].n_t;
            while (i + m < n && m < kMaxBatch && tot + c[i + m].n_t <= 0x7fff0000LL) { tot += c[i + m].n_t; ++m; }
        }
        // (what lies between two launches of this call is known: nothing)
        const filark_status_t st = launch_chunks(h, c.data() + i, m, stream, !first || (h->flags & FILARK_FLAG_OVERLAP_PUSHES) != 0);
        if (st != FILARK_OK) return st;
        first = false;
        i += m;
    }
    return FILARK_OK;
}

filark_status_t filark_stream_push_host(filark_stream_t* h, const float* h_in, long long n_t,
                                        float* h_filt, float* h_cf, cudaStream_t stream)
{
    if (!h || n_t < 0) return FILARK_ERR_INVALID_ARG;
    if (n_t == 0) return FILARK_OK;
    if (!h_in || (!h_filt && !h_cf)) return FILARK_ERR_INVALID_ARG;
    const size_t elems = (size_t)h->n_ch * (size_t)n_t;
    // (streams, events and staging buffers belong to the handle's device)
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(h, e);
    if (dev != h->device) return FILARK_ERR_DEVICE_MISMATCH;
    if (!h->host_ready) {
        e = cudaStreamCreateWithFlags(&h->s_h2d, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->s_d2h, cudaStreamNonBlocking);
        for (int j = 0; j < 2 && e == cudaSuccess; ++j) {
            e = cudaEventCreateWithFlags(&h->ev_h2d[j], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_kernel[j], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_d2h[j], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) return cuda_fail(h, e);
        h->host_ready = true;
    }
    if (elems > h->stage_elems) {
        cudaStreamSynchronize(stream); cudaStreamSynchronize(h->s_h2d); cudaStreamSynchronize(h->s_d2h);
        for (int j = 0; j < 2; ++j) for (int i = 0; i < 3; ++i) { cudaFree(h->d_stage[j][i]); h->d_stage[j][i] = nullptr; }
        h->stage_elems = 0;
        for (int j = 0; j < 2; ++j)
            for (int i = 0; i < 3 && e == cudaSuccess; ++i)
                e = cudaMalloc((void**)&h->d_stage[j][i], sizeof(float) * elems);
        if (e != cudaSuccess) {
            for (int j = 0; j < 2; ++j) for (int i = 0; i < 3; ++i) { cudaFree(h->d_stage[j][i]); h->d_stage[j][i] = nullptr; }
            cudaGetLastError();
            h->last_cuda_error = (int)e;
            return e == cudaErrorMemoryAllocation ? FILARK_ERR_ALLOC : FILARK_ERR_CUDA;
        }
        h->stage_elems = elems;
        h->ev_pending[0] = h->ev_pending[1] = false;
    }
    // Upload on the handle's upload stream, kernel on the caller's stream, download on the handle's
    // download stream: the upload of this chunk overlaps the download of the one before it (PCIe is
    // full duplex).  The caller's stream waits for the download at the end, so that synchronising
    // it still means "outputs are in host memory".
    const int j = (int)(h->host_pushes & 1u);
    float* const* st = h->d_stage[j];
    if (h->ev_pending[j]) {
        // set j was last used two pushes ago: its kernel must have read the input buffer, its
        // download must have read the output buffers
        e = cudaStreamWaitEvent(h->s_h2d, h->ev_kernel[j], 0);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, h->ev_d2h[j], 0);
        if (e != cudaSuccess) return cuda_fail(h, e);
    }
    e = cudaMemcpyAsync(st[0], h_in, sizeof(float) * elems, cudaMemcpyHostToDevice, h->s_h2d);
    if (e == cudaSuccess) e = cudaEventRecord(h->ev_h2d[j], h->s_h2d);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, h->ev_h2d[j], 0);
    if (e != cudaSuccess) return cuda_fail(h, e);
    const filark_status_t stt = filark_stream_push(h, st[0], n_t, h_filt ? st[1] : nullptr, h_cf ? st[2] : nullptr, stream);
    if (stt != FILARK_OK) return stt;
    e = cudaEventRecord(h->ev_kernel[j], stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(h->s_d2h, h->ev_kernel[j], 0);
    if (e == cudaSuccess && h_filt)
        e = cudaMemcpyAsync(h_filt, st[1], sizeof(float) * elems, cudaMemcpyDeviceToHost, h->s_d2h);
    if (e == cudaSuccess && h_cf)
        e = cudaMemcpyAsync(h_cf, st[2], sizeof(float) * elems, cudaMemcpyDeviceToHost, h->s_d2h);
    if (e == cudaSuccess) e = cudaEventRecord(h->ev_d2h[j], h->s_d2h);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, h->ev_d2h[j], 0);
    if (e != cudaSuccess) return cuda_fail(h, e);
    h->ev_pending[j] = true;
    h->host_pushes += 1;
    return FILARK_OK;
}

// ---- trigger / event emission on the characteristic function -------------
filark_status_t filark_stream_set_trigger(filark_stream_t* h, float thr_on, float thr_off, long long max_events,
                                          cudaStream_t stream)
{
    if (!h) return FILARK_ERR_INVALID_ARG;
    if (h->flags & FILARK_FLAG_SERIAL_SCAN) return FILARK_ERR_INVALID_ARG;
    const bool off = thr_on == 0.0f && thr_off == 0.0f;
    if (!off && (!(thr_on > 0.0f) || !(thr_off > 0.0f) || thr_off > thr_on || !std::isfinite(thr_on) ||
                 max_events < 1 || max_events > 0x7fffffffLL))
        return FILARK_ERR_INVALID_ARG;
    filark_status_t st = check_device(h);
    if (st != FILARK_OK) return st;
    // everything enqueued so far runs with the old settings
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return cuda_fail(h, e);
    if (!off && (unsigned)max_events != h->ev_cap) {
        cudaFree(h->d_events); h->d_events = nullptr; h->ev_cap = 0;
        e = cudaMalloc((void**)&h->d_events, sizeof(Event) * (size_t)max_events);
        if (e != cudaSuccess) { cudaGetLastError(); h->last_cuda_error = (int)e; h->thr_on = h->thr_off = 0.0f; return FILARK_ERR_ALLOC; }
        h->ev_cap = (unsigned)max_events;
    }
    if (!h->d_n_events) {
        e = cudaMalloc((void**)&h->d_n_events, sizeof(unsigned));
        if (e != cudaSuccess) { cudaGetLastError(); h->last_cuda_error = (int)e; return FILARK_ERR_ALLOC; }
    }
    // no event pending, every channel off
    e = cudaMemset(h->d_n_events, 0, sizeof(unsigned));
    const int ns = state_floats(h->n_sec);
    if (e == cudaSuccess)
        e = cudaMemset2D(h->d_state + trig_word(h->n_sec), sizeof(float) * (size_t)ns, 0, sizeof(float) * kTrigWords, (size_t)h->n_ch);
    if (e != cudaSuccess) return cuda_fail(h, e);
    h->thr_on = off ? 0.0f : thr_on; h->thr_off = off ? 0.0f : thr_off;
    return FILARK_OK;
}

filark_status_t filark_stream_pop_events(filark_stream_t* h, filark_event_t* out, long long cap, long long* n_out,
                                         long long* n_dropped, cudaStream_t stream)
{
    if (!h || !n_out || cap < 0 || (cap > 0 && !out)) return FILARK_ERR_INVALID_ARG;
    *n_out = 0;
    if (n_dropped) *n_dropped = 0;
    if (!h->d_n_events) return FILARK_OK;                      // no trigger was ever set
    filark_status_t st = check_device(h);
    if (st != FILARK_OK) return st;
    cudaError_t e = cudaStreamSynchronize(stream);
    unsigned n = 0;
    if (e == cudaSuccess) e = cudaMemcpy(&n, h->d_n_events, sizeof(n), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(h, e);
    const unsigned kept = n < h->ev_cap ? n : h->ev_cap;
    *n_out = (long long)kept;
    if (n_dropped) *n_dropped = (long long)(n - kept);
    if ((long long)kept > cap) return FILARK_ERR_INVALID_ARG;   // nothing consumed: call again with room for *n_out events
    static_assert(sizeof(filark_event_t) == sizeof(Event), "event record");
    if (kept) e = cudaMemcpy(out, h->d_events, sizeof(Event) * (size_t)kept, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemset(h->d_n_events, 0, sizeof(unsigned));
    if (e != cudaSuccess) return cuda_fail(h, e);
    return FILARK_OK;
}

// ---- zero-phase window mode (reading R29) -----------------------
// state[c][i] = kvec[i] * (first sample of channel c): the steady state of the cascade for that level
struct IcParams { float kvec[2 * kMaxSec]; };
__global__ void filark_ic_kernel(float* state, int ns, int n_state, const __grid_constant__ IcParams k,
                                 const float* x, long long stride_c, int n_ch)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_ch) return;
    const float x0 = x[(long long)c * stride_c];
    for (int i = 0; i < n_state; ++i) state[(long long)c * ns + i] = k.kvec[i] * x0;
}
// out(c, n) = in(c, n_t - 1 - n); element (c, n) at c*sc + n*sn
__global__ void filark_reverse_kernel(const float* in, float* out, int n_ch, long long n_t, long long sc, long long sn, int fast_c)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)n_ch * n_t) return;
    // consecutive threads along the contiguous axis of the layout
    const long long c = fast_c ? i % n_ch : i / n_t, n = fast_c ? i / n_ch : i % n_t;
    out[c * sc + n * sn] = in[c * sc + (n_t - 1 - n) * sn];
}

filark_status_t filark_stream_zero_phase(filark_stream_t* h, const float* d_in, long long n_t, float* d_out, cudaStream_t stream)
{
    if (!h || n_t < 0) return FILARK_ERR_INVALID_ARG;
    if (n_t == 0) return FILARK_OK;
    if (!d_in || !d_out || n_t > 0x7fff0000LL || (h->flags & FILARK_FLAG_SERIAL_SCAN)) return FILARK_ERR_INVALID_ARG;
    if (((uintptr_t)d_in | (uintptr_t)d_out) & 3u) return FILARK_ERR_ALIGNMENT;
    filark_status_t st = check_device(h);
    if (st != FILARK_OK) return st;
    const size_t elems = (size_t)h->n_ch * (size_t)n_t;
    if (!h->zp) {
        st = filark_stream_create_ex(&h->zp, h->n_ch, h->sos, h->n_sec, 1, 1, h->layout, FILARK_FLAG_NONE);
        if (st != FILARK_OK) { h->zp = nullptr; return st; }
    }
    if (elems > h->zp_elems) {
        cudaStreamSynchronize(stream);
        cudaDeviceSynchronize();
        cudaFree(h->d_zp_tmp[0]); cudaFree(h->d_zp_tmp[1]);
        h->d_zp_tmp[0] = h->d_zp_tmp[1] = nullptr; h->zp_elems = 0;
        cudaError_t e = cudaMalloc((void**)&h->d_zp_tmp[0], sizeof(float) * elems);
        if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_zp_tmp[1], sizeof(float) * elems);
        if (e != cudaSuccess) {
            cudaFree(h->d_zp_tmp[0]); cudaFree(h->d_zp_tmp[1]); h->d_zp_tmp[0] = h->d_zp_tmp[1] = nullptr;
            cudaGetLastError(); h->last_cuda_error = (int)e;
            return e == cudaErrorMemoryAllocation ? FILARK_ERR_ALLOC : FILARK_ERR_CUDA;
        }
        h->zp_elems = elems;
    }
    // steady state of the cascade per unit input level (float64, as filark_stream_set_initial_condition)
    filark_stream* z = h->zp;
    IcParams k{};
    {
        double v = z->gain;
        for (int j = 0; j < z->n_sec; ++j) {
            const Section& q = z->sec[j];
            const double m00 = 1.0 - q.A.a, m01 = -q.A.b, m10 = -q.A.c, m11 = 1.0 - q.A.d;
            const double det = m00 * m11 - m01 * m10, b0 = q.B[0] * v, b1 = q.B[1] * v;
            const double s0 = (m11 * b0 - m01 * b1) / det, s1 = (m00 * b1 - m10 * b0) / det;
            k.kvec[2 * j] = (float)s0; k.kvec[2 * j + 1] = (float)s1;
            v = q.C[0] * s0 + q.C[1] * s1 + q.D * v;
        }
    }
    const bool cm = h->layout == FILARK_LAYOUT_CHANNEL_MAJOR;
    const long long sc = cm ? n_t : 1, sn = cm ? 1 : (long long)h->n_ch;
    const int ns = state_floats(h->n_sec);
    const unsigned gc = (unsigned)((h->n_ch + 127) / 128), ge = (unsigned)((elems + 255) / 256);
    const float* src = d_in;
    for (int pass = 0; pass < 2; ++pass) {
        st = filark_stream_reset(z, stream);
        if (st != FILARK_OK) return st;
        filark_ic_kernel<<<gc, 128, 0, stream>>>(z->d_state, ns, 2 * h->n_sec, k, src, sc, h->n_ch);
        st = filark_stream_push(z, src, n_t, h->d_zp_tmp[0], nullptr, stream);
        if (st != FILARK_OK) return st;
        float* dst = pass == 0 ? h->d_zp_tmp[1] : d_out;
        filark_reverse_kernel<<<ge, 256, 0, stream>>>(h->d_zp_tmp[0], dst, h->n_ch, n_t, sc, sn, cm ? 0 : 1);
        src = h->d_zp_tmp[1];
    }
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? FILARK_OK : cuda_fail(h, e);
}

// ---- state export / import, initial condition ----------------------------
// Documented form (include/filark_stream.h): header + per channel 2 n_sec + 2 doubles = the state s
// of every section in the coordinates of filark_debug_design (s[n] = A s[n-1] + B x[n], the cascade's
// gain applied in front of section 0) after the LAST pushed sample, then sta N_s and lta N_l.
struct StateHeader {
    char magic[8];                 // "FKSTATE1"
    int n_ch, n_sec, sta_len, lta_len;
    unsigned long long seen;       // samples per channel since create/reset
    unsigned char pad[32];
};
static_assert(sizeof(StateHeader) == 64, "blob header");

long long filark_stream_state_size(const filark_stream_t* h)
{
    return h ? (long long)sizeof(StateHeader) + (long long)h->n_ch * (2LL * h->n_sec + 2) * (long long)sizeof(double) : -1;
}

// (host, float64) one sample through the conditioned cascade and the averages, as the kernels run them
static void host_step(const filark_stream* h, double* s, double x)
{
    double v = h->gain * x;
    for (int k = 0; k < h->n_sec; ++k) {
        const Section& c = h->sec[k];
        double* q = s + 2 * k;
        const double y = c.C[0] * q[0] + c.C[1] * q[1] + c.D * v;
        const double n0 = c.A.a * q[0] + c.A.b * q[1] + c.B[0] * v;
        const double n1 = c.A.c * q[0] + c.A.d * q[1] + c.B[1] * v;
        q[0] = n0; q[1] = n1;
        v = y;
    }
    const double e = v * v;
    double* m = s + 2 * h->n_sec;
    m[0] = m[0] - m[0] / h->sta_len + e;          // m~ = N m:  m~ <- (1 - 1/N) m~ + e
    m[1] = m[1] - m[1] / h->lta_len + e;
}

filark_status_t filark_stream_get_state(filark_stream_t* h, void* blob, long long size, cudaStream_t stream)
{
    if (!h || !blob || size < filark_stream_state_size(h)) return FILARK_ERR_INVALID_ARG;
    if (h->flags & FILARK_FLAG_SERIAL_SCAN) return FILARK_ERR_INVALID_ARG;
    filark_status_t st = check_device(h);
    if (st != FILARK_OK) return st;
    const int ns = state_floats(h->n_sec), w = 2 * h->n_sec + 2;
    std::vector<float> state((size_t)h->n_ch * ns), hist((size_t)h->n_ch * kHist);
    CmCtl ctl;
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();           // (pushes of this handle on other streams)
    if (e == cudaSuccess) e = cudaMemcpy(state.data(), h->d_state, sizeof(float) * state.size(), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(hist.data(), h->d_hist, sizeof(float) * hist.size(), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(&ctl, h->d_cctl, sizeof(ctl), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(h, e);
    const CmSlot& sl = ctl.slot[ctl.epoch & 1u];
    StateHeader hd{};
    std::memcpy(hd.magic, "FKSTATE1", 8);
    hd.n_ch = h->n_ch; hd.n_sec = h->n_sec; hd.sta_len = h->sta_len; hd.lta_len = h->lta_len;
    hd.seen = sl.seen;
    std::memcpy(blob, &hd, sizeof(hd));
    double* out = reinterpret_cast<double*>(static_cast<char*>(blob) + sizeof(hd));
    // the device state stands at the last slot boundary: run the r0 samples waiting in `hist` over it
    const int r0 = (int)sl.r0 < kHist ? (int)sl.r0 : kHist - 1;
    for (int c = 0; c < h->n_ch; ++c) {
        double* s = out + (size_t)c * w;
        for (int i = 0; i < w; ++i) s[i] = (double)state[(size_t)c * ns + i];
        for (int j = 0; j < r0; ++j) host_step(h, s, (double)hist[(size_t)c * kHist + j]);
    }
    return FILARK_OK;
}

// state words of every channel (float64, documented coordinates) -> handle, `seen` samples on the counter
static filark_status_t install_state(filark_stream_t* h, const double* in, unsigned long long seen, cudaStream_t stream)
{
    const int ns = state_floats(h->n_sec), w = 2 * h->n_sec + 2;
    std::vector<float> state((size_t)h->n_ch * ns, 0.0f);
    for (int c = 0; c < h->n_ch; ++c)
        for (int i = 0; i < w; ++i) state[(size_t)c * ns + i] = (float)in[(size_t)c * w + i];
    CmCtl ctl;
    std::memset(&ctl, 0, sizeof(ctl));
    ctl.slot[0].seen = seen;
    cudaError_t e = cudaStreamSynchronize(stream);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(h->d_state, state.data(), sizeof(float) * state.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(h->d_hist, 0, sizeof(float) * (size_t)h->n_ch * kHist);
    if (e == cudaSuccess) e = cudaMemcpy(h->d_cctl, &ctl, sizeof(ctl), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(h->d_progress, 0, sizeof(unsigned) * (size_t)h->n_ch);
    if (e != cudaSuccess) return cuda_fail(h, e);
    h->prev_valid = 0;
    h->samples = (long long)seen;
    return FILARK_OK;
}

filark_status_t filark_stream_set_state(filark_stream_t* h, const void* blob, long long size, cudaStream_t stream)
{
    if (!h || !blob || size < filark_stream_state_size(h)) return FILARK_ERR_INVALID_ARG;
    if (h->flags & FILARK_FLAG_SERIAL_SCAN) return FILARK_ERR_INVALID_ARG;
    StateHeader hd;
    std::memcpy(&hd, blob, sizeof(hd));
    if (std::memcmp(hd.magic, "FKSTATE1", 8) != 0 || hd.n_ch != h->n_ch || hd.n_sec != h->n_sec ||
        hd.sta_len != h->sta_len || hd.lta_len != h->lta_len)
        return FILARK_ERR_INVALID_ARG;
    const int w = 2 * h->n_sec + 2;
    const double* in = reinterpret_cast<const double*>(static_cast<const char*>(blob) + sizeof(hd));
    for (long long i = 0; i < (long long)h->n_ch * w; ++i) if (!std::isfinite(in[i])) return FILARK_ERR_INVALID_ARG;
    filark_status_t st = check_device(h);
    if (st != FILARK_OK) return st;
    return install_state(h, in, hd.seen, stream);
}

filark_status_t filark_stream_set_initial_condition(filark_stream_t* h, const float* x0, cudaStream_t stream)
{
    if (!h || !x0) return FILARK_ERR_INVALID_ARG;
    if (h->flags & FILARK_FLAG_SERIAL_SCAN) return FILARK_ERR_INVALID_ARG;
    for (int c = 0; c < h->n_ch; ++c) if (!std::isfinite(x0[c])) return FILARK_ERR_INVALID_ARG;
    filark_status_t st = check_device(h);
    if (st != FILARK_OK) return st;
    // steady state of s = A s + B v, y = C s + D v for a constant input v: s = (I - A)^-1 B v
    const int w = 2 * h->n_sec + 2;
    std::vector<double> in((size_t)h->n_ch * w);
    for (int c = 0; c < h->n_ch; ++c) {
        double v = h->gain * (double)x0[c];
        double* s = in.data() + (size_t)c * w;
        for (int k = 0; k < h->n_sec; ++k) {
            const Section& q = h->sec[k];
            const double m00 = 1.0 - q.A.a, m01 = -q.A.b, m10 = -q.A.c, m11 = 1.0 - q.A.d;
            const double det = m00 * m11 - m01 * m10;                 // = 1 + a1 + a2 > 0 (stable section)
            const double b0 = q.B[0] * v, b1 = q.B[1] * v;
            s[2 * k] = (m11 * b0 - m01 * b1) / det;
            s[2 * k + 1] = (m00 * b1 - m10 * b0) / det;
            v = q.C[0] * s[2 * k] + q.C[1] * s[2 * k + 1] + q.D * v;
        }
        s[2 * h->n_sec] = v * v * h->sta_len;
        s[2 * h->n_sec + 1] = v * v * h->lta_len;
    }
    return install_state(h, in.data(), (unsigned long long)h->lta_len, stream);
}

// ---- debug / introspection (include/filark_debug.h): host only, no CUDA calls -----------------
int filark_debug_design(const double* sos, int n_sec, int* kinds, double* coefs, double* gain)
{
    if (!sos || n_sec <= 0 || n_sec > FILARK_MAX_SECTIONS) return (int)FILARK_ERR_INVALID_ARG;
    Section sec[kMaxSec];
    double g = 1.0;
    const filark_status_t st = design_all(sos, n_sec, sec, &g);
    if (st != FILARK_OK) return (int)st;
    for (int k = 0; k < n_sec; ++k) {
        if (kinds) kinds[k] = sec[k].kind;
        if (coefs) {
            double* c = coefs + 9 * k;      // A (4, row-major), B (2), C (2), D
            c[0] = sec[k].A.a; c[1] = sec[k].A.b; c[2] = sec[k].A.c; c[3] = sec[k].A.d;
            c[4] = sec[k].B[0]; c[5] = sec[k].B[1]; c[6] = sec[k].C[0]; c[7] = sec[k].C[1];
            c[8] = sec[k].D;
        }
    }
    if (gain) *gain = g;
    return (int)FILARK_OK;
}

int filark_debug_push_geometry(long long n_t, int r0, int force_L, int* out5)
{
    if (n_t < 1 || n_t > 0x7fff0000LL || r0 < 0 || r0 >= kHist || !out5) return (int)FILARK_ERR_INVALID_ARG;
    int L = 0;
    if (force_L == 0) L = kVariantL[choose_variant(n_t)];
    else for (int v = 0; v < kNumVariants; ++v) if (kVariantL[v] == force_L) L = force_L;
    if (L == 0) return (int)FILARK_ERR_INVALID_ARG;
    const Geom g = geometry_rt(L, (unsigned)r0, (int)n_t, true);
    out5[0] = L; out5[1] = g.n_tiles; out5[2] = g.q_last; out5[3] = g.r1; out5[4] = g.vec4 ? 1 : 0;
    return (int)FILARK_OK;
}

int filark_debug_block_power(const double* sos6, long long e, double* out4)
{
    if (!sos6 || !out4 || e < 0) return (int)FILARK_ERR_INVALID_ARG;
    Section s;
    const DesignStatus ds = design_section(sos6, &s);
    if (ds != DESIGN_OK) return ds == DESIGN_UNSTABLE ? (int)FILARK_ERR_UNSTABLE : (int)FILARK_ERR_INVALID_ARG;
    const Mat2 m = mpow(s.A, e);
    out4[0] = m.a; out4[1] = m.b; out4[2] = m.c; out4[3] = m.d;
    return (int)FILARK_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------
// filark_stream_once_noalloc (include/filark_stream.h): the push kernel over one record from rest, with
// the device memory a handle would own -- carried state, raw-history rows, progress words, control block --
// in ONE fixed array of the library's device image instead of cudaMalloc'ed buffers.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address: the address
// the kernel gets comes from cudaGetSymbolAddress, asked once per device with that device current.
namespace {

constexpr int kNaMaxCh = FILARK_NOALLOC_MAX_CHANNELS;
constexpr size_t kNaStateBytes = sizeof(float) * (size_t)kNaMaxCh * (size_t)state_floats(kMaxSec);
constexpr size_t kNaHistBytes = sizeof(float) * (size_t)kNaMaxCh * (size_t)kHist;
constexpr size_t kNaProgressBytes = sizeof(unsigned) * (size_t)kNaMaxCh;
constexpr size_t kNaHistOff = kNaStateBytes, kNaProgressOff = kNaHistOff + kNaHistBytes, kNaCtlOff = kNaProgressOff + kNaProgressBytes;
constexpr size_t kNaBytes = kNaCtlOff + 256;
static_assert(kNaBytes == (size_t)FILARK_NOALLOC_SCRATCH_BYTES, "the header states the size of the array");
static_assert(kNaHistOff % 256 == 0 && kNaProgressOff % 256 == 0 && kNaCtlOff % 256 == 0 && sizeof(CmCtl) <= 256, "aligned parts");

static __device__ __align__(256) unsigned char fk_noalloc_scratch[kNaBytes];

std::mutex g_na_mutex;
unsigned char* g_na_ptr[kMaxDevices];       // device address of fk_noalloc_scratch, by device

// Device address of the array on the CURRENT device (`device`).
cudaError_t noalloc_scratch(int device, unsigned char** out)
{
    const bool tracked = device >= 0 && device < kMaxDevices;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (tracked && g_na_ptr[device]) { *out = g_na_ptr[device]; return cudaSuccess; }
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, fk_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!ptr) return cudaErrorInvalidSymbol;
    if (tracked) g_na_ptr[device] = (unsigned char*)ptr;
    *out = (unsigned char*)ptr;
    return cudaSuccess;
}

// "the last launch on this stream was not yours", for every handle (registry_is_last): a handle that pushes
// behind this call in the same stream must not let its push start early
const filark_stream* const kNaForeign = reinterpret_cast<const filark_stream*>(&g_na_mutex);

}  // namespace

extern "C" filark_status_t filark_stream_once_noalloc(const double* sos, int n_sec, int sta_len, int lta_len, int layout,
                                                      const float* d_in, int n_ch, long long n_t, float* d_filt,
                                                      float* d_cf, cudaStream_t stream, int* cuda_error)
{
    if (cuda_error) *cuda_error = 0;
    auto fail = [&](cudaError_t e) { if (cuda_error) *cuda_error = (int)e; cudaGetLastError(); return FILARK_ERR_CUDA; };
    filark_status_t st = check_create_args(&st, n_ch, sos, n_sec, sta_len, lta_len, layout, FILARK_FLAG_NONE);
    if (st != FILARK_OK) return st;
    if (n_t < 0) return FILARK_ERR_INVALID_ARG;
    if (n_ch > kNaMaxCh) return FILARK_ERR_TOO_LARGE;
    if (n_t == 0) return FILARK_OK;

    // a handle on the stack: the design of the cascade and what the launch code reads of a handle
    filark_stream h;
    std::memset(&h, 0, sizeof(h));
    st = design_all(sos, n_sec, h.sec, &h.gain);
    if (st != FILARK_OK) return st;
    h.lean_kinds = !tune().all_kinds;
    for (int k = 0; k < n_sec; ++k) h.lean_kinds = h.lean_kinds && (h.sec[k].kind == kKindDF2 || h.sec[k].kind == kKindDelta);
    h.n_ch = n_ch; h.n_sec = n_sec; h.sta_len = sta_len; h.lta_len = lta_len; h.layout = layout; h.flags = FILARK_FLAG_NONE;
    h.state_floats = (size_t)n_ch * (size_t)state_floats(n_sec);

    const long long pitch = layout == FILARK_LAYOUT_CHANNEL_MAJOR ? n_t : (long long)n_ch;
    const ChunkArgs c{d_in, n_t, pitch, d_filt, d_cf, pitch};
    size_t ib = 0, ob = 0;
    st = check_chunk(&h, c, &ib, &ob);
    if (st != FILARK_OK) return st;

    cudaError_t e = cudaGetDevice(&h.device);
    int optin = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h.n_sm, cudaDevAttrMultiProcessorCount, h.device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h.device);
    h.smem_optin = (size_t)optin;
    unsigned char* base = nullptr;
    if (e == cudaSuccess) e = noalloc_scratch(h.device, &base);
    if (e != cudaSuccess) return fail(e);
    h.d_state = reinterpret_cast<float*>(base);
    h.d_hist = reinterpret_cast<float*>(base + kNaHistOff);
    h.d_progress = reinterpret_cast<unsigned*>(base + kNaProgressOff);
    h.d_cctl = reinterpret_cast<CmCtl*>(base + kNaCtlOff);

    // the array keeps what the last call left: from rest means state, progress and control block at zero
    // (the history rows are read only as far as the control block says, i.e. not at all)
    e = cudaMemsetAsync(h.d_state, 0, sizeof(float) * h.state_floats, stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h.d_progress, 0, sizeof(unsigned) * (size_t)n_ch, stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h.d_cctl, 0, sizeof(CmCtl), stream);
    if (e != cudaSuccess) return fail(e);

    // tables of the one variant this record takes, on the stack
    // (time-major: the kernel with one channel per lane, as a handle without a trigger takes it)
    const bool cm = layout == FILARK_LAYOUT_CHANNEL_MAJOR;
    const bool lanes = !cm && pitch < (1LL << 25) && n_t >= 4LL * kTrRows;
    int v = choose_variant(n_t);
    if (lanes) for (int i = 0; i < kNumVariants; ++i) if (kVariantL[i] == kTrL) v = i;
    alignas(16) unsigned char proto[sizeof(PushParams<24>)];
    static_assert(sizeof(PushParams<24>) >= sizeof(PushParams<16>) && sizeof(PushParams<24>) >= sizeof(PushParams<8>), "largest variant");
    h.proto[v] = proto;
    const uintptr_t all = (uintptr_t)d_in | (uintptr_t)d_filt | (uintptr_t)d_cf;
    const int vec4 = cm ? ((all & 15u) == 0 && (n_t & 3) == 0) : ((((uintptr_t)d_filt | (uintptr_t)d_cf) & 15u) == 0 && (n_ch & 3) == 0);
    switch (kVariantL[v]) {
        case 8: build_proto<8>(&h, reinterpret_cast<PushParams<8>*>(proto)); e = push_variant<8>(&h, v, &c, 1, vec4, 1, stream); break;
        case 16: build_proto<16>(&h, reinterpret_cast<PushParams<16>*>(proto)); e = push_variant<16>(&h, v, &c, 1, vec4, 1, stream); break;
        default: build_proto<24>(&h, reinterpret_cast<PushParams<24>*>(proto)); e = push_variant<24>(&h, v, &c, 1, vec4, 1, stream, lanes); break;
    }
    registry_set(stream, kNaForeign);
    if (e != cudaSuccess) return fail(e);
    return FILARK_OK;
}

// ---------------------------------------------------------------------------------------------------
// filark_events_associate (include/filark_stream.h; reading R30): host work on a host list.
extern "C" filark_status_t filark_events_associate(const filark_event_t* ev, long long n, int ch_gap, long long t_gap,
                                                   filark_box_t* boxes, long long cap, long long* n_boxes)
{
    if (!n_boxes || n < 0 || cap < 0 || ch_gap < 0 || t_gap < 0 || (n > 0 && !ev) || (cap > 0 && !boxes) || n > 0x7fffffffLL)
        return FILARK_ERR_INVALID_ARG;
    *n_boxes = 0;
    if (n == 0) return FILARK_OK;
    try {
        const int m = (int)n;
        std::vector<int> order(m), parent(m);
        for (int i = 0; i < m; ++i) order[i] = parent[i] = i;
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return ev[a].t_on < ev[b].t_on; });
        auto find = [&](int i) { while (parent[i] != i) { parent[i] = parent[parent[i]]; i = parent[i]; } return i; };
        // events still within reach of a later one, by channel.  In rising t_on an event j is out of reach
        // for good once t_off[j] + t_gap <= t_on of the event at hand.
        std::map<int, std::vector<int>> active;
        for (int oi = 0; oi < m; ++oi) {
            const int i = order[oi];
            const filark_event_t& e = ev[i];
            const long long lo = (long long)e.channel - ch_gap, hi = (long long)e.channel + ch_gap;
            for (auto it = active.lower_bound((int)std::max(lo, (long long)INT32_MIN)); it != active.end() && it->first <= hi;) {
                std::vector<int>& v = it->second;
                size_t keep = 0;
                for (size_t q = 0; q < v.size(); ++q) {
                    const filark_event_t& o = ev[v[q]];
                    if (o.t_off + t_gap <= e.t_on) continue;                     // out of reach for good
                    v[keep++] = v[q];
                    if (o.t_on < e.t_off + t_gap) { const int a = find(i), b = find(v[q]); if (a != b) parent[a] = b; }
                }
                v.resize(keep);
                if (v.empty()) it = active.erase(it); else ++it;
            }
            active[e.channel].push_back(i);
        }
        std::vector<int> box_of(m, -1);
        std::vector<filark_box_t> out;
        for (int i = 0; i < m; ++i) {
            const int r = find(i);
            const filark_event_t& e = ev[i];
            if (box_of[r] < 0) {
                box_of[r] = (int)out.size();
                out.push_back(filark_box_t{e.t_on, e.t_off, e.channel, e.channel, e.peak, 1});
            } else {
                filark_box_t& b = out[(size_t)box_of[r]];
                b.t_on = std::min(b.t_on, e.t_on); b.t_off = std::max(b.t_off, e.t_off);
                b.ch_lo = std::min(b.ch_lo, e.channel); b.ch_hi = std::max(b.ch_hi, e.channel);
                b.peak = std::max(b.peak, e.peak); b.n_events += 1;
            }
        }
        std::stable_sort(out.begin(), out.end(), [](const filark_box_t& a, const filark_box_t& b) {
            if (a.t_on != b.t_on) return a.t_on < b.t_on;
            if (a.ch_lo != b.ch_lo) return a.ch_lo < b.ch_lo;
            if (a.t_off != b.t_off) return a.t_off < b.t_off;
            return a.ch_hi < b.ch_hi;
        });
        *n_boxes = (long long)out.size();
        const size_t w = std::min((size_t)cap, out.size());
        for (size_t i = 0; i < w; ++i) boxes[i] = out[i];
    } catch (const std::bad_alloc&) {
        return FILARK_ERR_ALLOC;
    }
    return FILARK_OK;
}
