// filark_stream.cu -- C ABI (include/filark_stream.h) + host-side preparation + launches.
//
// Host work per create: validate, rewrite every SOS section as a conditioned 2-state system
// (design.hpp), build the float64 block-power / fix-up tables, round to fp32, upload, zero the
// carried state.  Host work per push: argument checks, the tail-tile table for this n_t
// (cached), ONE kernel launch on the caller's stream.  No synchronisation, no allocation.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/filark_stream.h"
#include "../../include/filark_debug.h"
#include "design.hpp"
#include "filark_kernels.cuh"

using namespace filark;

// Sub-block lengths compiled as kernel variants; a push picks the cheapest for its n_t.
static const int kVariantL[] = {8, 16, 24, 32, 48};
constexpr int kNumVariants = 5;

struct Geometry { int L, n_tiles, lead, r, pad0, last_lane, last_half; };

struct filark_stream {
    int device;
    int n_ch, n_sec, sta_len, lta_len, layout;
    unsigned flags;
    Section sec[kMaxSec];
    double gain;
    float* d_tab[kNumVariants];
    size_t tab_floats[kNumVariants];
    float* d_state;
    size_t state_floats;
    int n_sm;
    size_t smem_optin;
    int last_cuda_error;
    long long launches, samples;
    // staging for push_host
    float* d_stage[3];
    size_t stage_elems;
};

static filark_status_t cuda_fail(filark_stream* h, cudaError_t e)
{
    if (h) h->last_cuda_error = (int)e;
    return FILARK_ERR_CUDA;
}

static void put_mat(float* dst, const Mat2& m)
{
    dst[0] = (float)m.a; dst[1] = (float)m.b; dst[2] = (float)m.c; dst[3] = (float)m.d;
}

template <int L> static size_t variant_floats(int n_sec)
{
    return (size_t)n_sec * SecTab<L>::stride + kAvgFloats;
}

// Device table of sub-block length L (layout documented in filark_kernels.cuh).
template <int L> static void build_variant_table(const filark_stream* h, float* tab)
{
    using ST = SecTab<L>;
    std::memset(tab, 0, sizeof(float) * variant_floats<L>(h->n_sec));
    for (int k = 0; k < h->n_sec; ++k) {
        const Section& s = h->sec[k];
        float* T = tab + (size_t)k * ST::stride;
        std::memcpy(&T[kOffKind], &s.kind, sizeof(int));
        for (int i = 0; i < 5; ++i) T[kOffCoef + i] = (float)s.coef[i];
        put_mat(T + kOffP, mpow(s.A, L));
        Mat2 q = mpow(s.A, 2 * L);
        int nsteps = kSteps;
        for (int d = 0; d < kSteps; ++d) {
            put_mat(T + kOffQ + 4 * d, q);
            if (nsteps == kSteps && norm1(q) < 1e-10) nsteps = d;      // this and later steps add < 1e-10
            q = mul(q, q);
        }
        std::memcpy(&T[kOffNSteps], &nsteps, sizeof(int));
        double g[2 * L];
        fixup_rows(s, L, g);
        for (int i = 0; i < L; ++i) {
            T[ST::g0 + 2 * (L + i)] = (float)g[2 * i];         T[ST::g0 + 2 * (L + i) + 1] = (float)g[2 * i + 1];
            T[ST::g1 + 2 * (L + i + 1)] = (float)g[2 * i];     T[ST::g1 + 2 * (L + i + 1) + 1] = (float)g[2 * i + 1];
        }
        // (row 2L of G1 would be g[L-1] shifted out of the table: it lands in the 4-float pad)
    }
    float* AV = tab + (size_t)h->n_sec * ST::stride;
    const double cs = 1.0 / h->sta_len, cl = 1.0 / h->lta_len;
    AV[0] = (float)(1.0 - cs); AV[1] = (float)(1.0 - cl);
    AV[kAvgBetaL] = (float)one_minus_pow(cs, L); AV[kAvgBetaL + 1] = (float)one_minus_pow(cl, L);
    for (int d = 0; d < kSteps; ++d) {
        const double e = 2.0 * L * (double)(1 << d);
        AV[kAvgBetaQ + 2 * d] = (float)one_minus_pow(cs, e);
        AV[kAvgBetaQ + 2 * d + 1] = (float)one_minus_pow(cl, e);
    }
    AV[kAvgInvN] = (float)cs; AV[kAvgInvN + 1] = (float)cl;
}

// What a push needs beyond the table: powers for its first (possibly short) slot of r samples.
static void fill_first_slot_params(const filark_stream* h, int L, int r, PushParams* p)
{
    const double cs = 1.0 / h->sta_len, cl = 1.0 / h->lta_len;
    const int sh = L - r;
    p->beta_r[0] = (float)one_minus_pow(cs, r); p->beta_r[1] = (float)one_minus_pow(cl, r);
    // alpha^-sh; alpha = 0 (length-1 average) keeps no memory, any finite factor will do
    p->inv_sh[0] = cs >= 1.0 ? (sh == 0 ? 1.0f : 0.0f) : (float)std::exp(-(double)sh * std::log1p(-cs));
    p->inv_sh[1] = cl >= 1.0 ? (sh == 0 ? 1.0f : 0.0f) : (float)std::exp(-(double)sh * std::log1p(-cl));
    for (int k = 0; k < h->n_sec; ++k) put_mat(&p->apow_r[k][0], mpow(h->sec[k].A, r));
}

static size_t variant_floats_rt(int v, int n_sec)
{
    switch (kVariantL[v]) {
        case 8: return variant_floats<8>(n_sec);
        case 16: return variant_floats<16>(n_sec);
        case 24: return variant_floats<24>(n_sec);
        case 32: return variant_floats<32>(n_sec);
        default: return variant_floats<48>(n_sec);
    }
}
static void build_variant_rt(int v, const filark_stream* h, float* tab)
{
    switch (kVariantL[v]) {
        case 8: build_variant_table<8>(h, tab); break;
        case 16: build_variant_table<16>(h, tab); break;
        case 24: build_variant_table<24>(h, tab); break;
        case 32: build_variant_table<32>(h, tab); break;
        default: build_variant_table<48>(h, tab); break;
    }
}
static int sec_stride_rt(int v)
{
    switch (kVariantL[v]) {
        case 8: return SecTab<8>::stride;
        case 16: return SecTab<16>::stride;
        case 24: return SecTab<24>::stride;
        case 32: return SecTab<32>::stride;
        default: return SecTab<48>::stride;
    }
}

// Slot geometry of a push of n_t >= 1 samples with sub-block length L: slots are aligned to the
// end of the push; a short first slot (r < L) sits behind one idle slot (high half of lane 0).
static Geometry geometry_for(long long n_t, int L)
{
    Geometry g{};
    g.L = L;
    const long long U = (n_t + L - 1) / L;                 // slots holding samples
    g.r = (int)(n_t - (U - 1) * L);
    g.lead = g.r < L ? 1 : 0;
    g.pad0 = g.lead * L + (L - g.r);
    const long long slots = U + g.lead;
    g.n_tiles = (int)((slots + 63) / 64);
    const int s_last = (int)((slots - 1) % 64);
    g.last_lane = s_last >> 1; g.last_half = s_last & 1;
    return g;
}

// Cheapest variant: a tile costs its L samples per lane-half plus a fixed part (scans, staging).
static int choose_variant(long long n_t)
{
    int best = 0; double best_cost = 1e300;
    for (int v = 0; v < kNumVariants; ++v) {
        const Geometry g = geometry_for(n_t, kVariantL[v]);
        const double cost = (double)g.n_tiles * (kVariantL[v] + 10.0);
        if (cost < best_cost) { best_cost = cost; best = v; }
    }
    return best;
}

// One CTA per SM; W warps per CTA as far as registers and shared memory allow; fewer, on more
// SMs, when there are few channels.
template <int L>
static cudaError_t launch_cm(const filark_stream* h, const PushParams& p, cudaStream_t stream)
{
    const size_t tab_bytes = sizeof(float) * variant_floats<L>(p.n_sec);
    const size_t warp_bytes = sizeof(float) * (size_t)warp_smem_floats<L>();
    int W = cm_max_warps<L>();
    const int fit = (int)((h->smem_optin - tab_bytes) / warp_bytes);
    if (fit < W) W = fit;
    const int want = (p.n_ch + h->n_sm - 1) / h->n_sm;
    if (want < W) W = want;
    if (W < 1) return cudaErrorInvalidConfiguration;
    const size_t smem = tab_bytes + (size_t)W * warp_bytes;
    static bool attr_done = false;           // per variant (template instance); idempotent
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(filark_push_cm_kernel<L>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)h->smem_optin);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    int grid = (p.n_ch + W - 1) / W;
    if (grid > h->n_sm) grid = h->n_sm;
    filark_push_cm_kernel<L><<<grid, W * 32, smem, stream>>>(p);
    return cudaGetLastError();
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
    if (flags & ~(FILARK_FLAG_SERIAL_SCAN | 0xFF00u)) return FILARK_ERR_INVALID_ARG;
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
    h->n_ch = n_ch; h->n_sec = n_sec; h->sta_len = sta_len; h->lta_len = lta_len;
    h->layout = layout; h->flags = flags;
    h->state_floats = (size_t)n_ch * (size_t)state_floats(n_sec);
    cudaError_t e = cudaGetDevice(&h->device);
    int optin = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    h->smem_optin = (size_t)optin;
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_state, sizeof(float) * h->state_floats);
    if (e == cudaSuccess) e = cudaMemset(h->d_state, 0, sizeof(float) * h->state_floats);
    bool host_oom = false;
    for (int v = 0; v < kNumVariants && e == cudaSuccess && !host_oom; ++v) {
        h->tab_floats[v] = variant_floats_rt(v, n_sec);
        float* tab = (float*)std::malloc(sizeof(float) * h->tab_floats[v]);
        if (!tab) { host_oom = true; break; }
        build_variant_rt(v, h, tab);
        e = cudaMalloc((void**)&h->d_tab[v], sizeof(float) * h->tab_floats[v]);
        if (e == cudaSuccess)
            e = cudaMemcpy(h->d_tab[v], tab, sizeof(float) * h->tab_floats[v], cudaMemcpyHostToDevice);
        std::free(tab);
    }
    if (e != cudaSuccess || host_oom) {
        const bool oom = host_oom || e == cudaErrorMemoryAllocation;
        for (int v = 0; v < kNumVariants; ++v) cudaFree(h->d_tab[v]);
        cudaFree(h->d_state);
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
    cudaDeviceSynchronize();
    for (int v = 0; v < kNumVariants; ++v) cudaFree(h->d_tab[v]);
    cudaFree(h->d_state);
    for (int i = 0; i < 3; ++i) cudaFree(h->d_stage[i]);
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
    if (e != cudaSuccess) return cuda_fail(h, e);
    h->samples = 0;
    return FILARK_OK;
}

static bool overlaps(const void* a, size_t na, const void* b, size_t nb)
{
    const uintptr_t a0 = (uintptr_t)a, b0 = (uintptr_t)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

filark_status_t filark_stream_push_pitched(filark_stream_t* h, const float* d_in, long long n_t,
                                           long long in_pitch, float* d_filt, float* d_cf,
                                           long long out_pitch, cudaStream_t stream)
{
    if (!h || n_t < 0) return FILARK_ERR_INVALID_ARG;
    if (n_t == 0) return FILARK_OK;
    if (!d_in || (!d_filt && !d_cf)) return FILARK_ERR_INVALID_ARG;
    const bool cm = h->layout == FILARK_LAYOUT_CHANNEL_MAJOR;
    const long long row_len = cm ? n_t : (long long)h->n_ch;
    const long long n_rows = cm ? (long long)h->n_ch : n_t;
    if (in_pitch < row_len || out_pitch < row_len) return FILARK_ERR_INVALID_ARG;
    if (((uintptr_t)d_in | (uintptr_t)d_filt | (uintptr_t)d_cf) & 3u) return FILARK_ERR_ALIGNMENT;
    const size_t in_bytes = sizeof(float) * (size_t)((n_rows - 1) * in_pitch + row_len);
    const size_t out_bytes = sizeof(float) * (size_t)((n_rows - 1) * out_pitch + row_len);
    if ((d_filt && overlaps(d_in, in_bytes, d_filt, out_bytes)) ||
        (d_cf && overlaps(d_in, in_bytes, d_cf, out_bytes)) ||
        (d_filt && d_cf && overlaps(d_filt, out_bytes, d_cf, out_bytes)))
        return FILARK_ERR_INVALID_ARG;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(h, e);
    if (dev != h->device) return FILARK_ERR_DEVICE_MISMATCH;

    PushParams p{};
    p.in = d_in; p.filt = d_filt; p.cf = d_cf;
    p.state = h->d_state;
    p.n_t = n_t; p.in_pitch = in_pitch; p.out_pitch = out_pitch;
    p.n_ch = h->n_ch; p.n_sec = h->n_sec;
    p.lta_len = h->lta_len;
    p.gain = (float)h->gain;
    p.ratio = (float)((double)h->lta_len / (double)h->sta_len);
    p.lta_thr = (float)(1e-30 * (double)h->lta_len);      // lta <= 1e-30  <=>  lta~ <= 1e-30 N_l
    const int ns = state_floats(h->n_sec);

    if ((h->flags & FILARK_FLAG_SERIAL_SCAN) || !cm) {
        // Serial diagnostic kernel; also the time-major path until the blocked time-major
        // kernel lands.
        const long long sc_in = cm ? in_pitch : 1, st_in = cm ? 1 : in_pitch;
        const long long sc_out = cm ? out_pitch : 1, st_out = cm ? 1 : out_pitch;
        const long long state_sc = cm ? ns : 1, state_sk = cm ? 1 : h->n_ch;
        const int block = 128, grid = (h->n_ch + block - 1) / block;
        p.tab = h->d_tab[0];
        filark_push_serial_kernel<<<grid, block, 0, stream>>>(p, sec_stride_rt(0), sc_in, st_in, sc_out,
                                                              st_out, state_sc, state_sk);
        e = cudaGetLastError();
    } else {
        int v = choose_variant(n_t);
        for (int i = 0; i < kNumVariants; ++i) if (kVariantL[i] == (int)((h->flags >> 8) & 0xFF)) v = i;
        const Geometry g = geometry_for(n_t, kVariantL[v]);
        p.tab = h->d_tab[v];
        p.n_tiles = g.n_tiles; p.lead = g.lead; p.r = g.r; p.pad0 = g.pad0;
        p.last_lane = g.last_lane; p.last_half = g.last_half;
        fill_first_slot_params(h, g.L, g.r, &p);
        const uintptr_t all = (uintptr_t)d_in | (uintptr_t)d_filt | (uintptr_t)d_cf;
        p.vec4 = ((all & 15u) == 0 && (in_pitch & 3) == 0 && (out_pitch & 3) == 0 && (n_t & 3) == 0) ? 1 : 0;
        switch (g.L) {
            case 8: e = launch_cm<8>(h, p, stream); break;
            case 16: e = launch_cm<16>(h, p, stream); break;
            case 24: e = launch_cm<24>(h, p, stream); break;
            case 32: e = launch_cm<32>(h, p, stream); break;
            default: e = launch_cm<48>(h, p, stream); break;
        }
    }
    if (e != cudaSuccess) return cuda_fail(h, e);
    h->launches += 1;
    h->samples += n_t;
    return FILARK_OK;
}

filark_status_t filark_stream_push(filark_stream_t* h, const float* d_in, long long n_t,
                                   float* d_filt, float* d_cf, cudaStream_t stream)
{
    if (!h) return FILARK_ERR_INVALID_ARG;
    const long long pitch = h->layout == FILARK_LAYOUT_CHANNEL_MAJOR ? n_t : (long long)h->n_ch;
    return filark_stream_push_pitched(h, d_in, n_t, pitch, d_filt, d_cf, pitch, stream);
}

filark_status_t filark_stream_push_host(filark_stream_t* h, const float* h_in, long long n_t,
                                        float* h_filt, float* h_cf, cudaStream_t stream)
{
    if (!h || n_t < 0) return FILARK_ERR_INVALID_ARG;
    if (n_t == 0) return FILARK_OK;
    if (!h_in || (!h_filt && !h_cf)) return FILARK_ERR_INVALID_ARG;
    const size_t elems = (size_t)h->n_ch * (size_t)n_t;
    cudaError_t e = cudaSuccess;
    if (elems > h->stage_elems) {
        cudaStreamSynchronize(stream);
        for (int i = 0; i < 3; ++i) { cudaFree(h->d_stage[i]); h->d_stage[i] = nullptr; }
        h->stage_elems = 0;
        for (int i = 0; i < 3 && e == cudaSuccess; ++i)
            e = cudaMalloc((void**)&h->d_stage[i], sizeof(float) * elems);
        if (e != cudaSuccess) {
            for (int i = 0; i < 3; ++i) { cudaFree(h->d_stage[i]); h->d_stage[i] = nullptr; }
            cudaGetLastError();
            h->last_cuda_error = (int)e;
            return e == cudaErrorMemoryAllocation ? FILARK_ERR_ALLOC : FILARK_ERR_CUDA;
        }
        h->stage_elems = elems;
    }
    e = cudaMemcpyAsync(h->d_stage[0], h_in, sizeof(float) * elems, cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) return cuda_fail(h, e);
    const filark_status_t st = filark_stream_push(h, h->d_stage[0], n_t, h_filt ? h->d_stage[1] : nullptr,
                                                  h_cf ? h->d_stage[2] : nullptr, stream);
    if (st != FILARK_OK) return st;
    if (h_filt) e = cudaMemcpyAsync(h_filt, h->d_stage[1], sizeof(float) * elems, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess && h_cf)
        e = cudaMemcpyAsync(h_cf, h->d_stage[2], sizeof(float) * elems, cudaMemcpyDeviceToHost, stream);
    if (e != cudaSuccess) return cuda_fail(h, e);
    return FILARK_OK;
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

int filark_debug_push_geometry(long long n_t, int force_L, int* out7)
{
    if (n_t < 1 || !out7) return (int)FILARK_ERR_INVALID_ARG;
    int L = 0;
    if (force_L == 0) L = kVariantL[choose_variant(n_t)];
    else for (int v = 0; v < kNumVariants; ++v) if (kVariantL[v] == force_L) L = force_L;
    if (L == 0) return (int)FILARK_ERR_INVALID_ARG;
    const Geometry g = geometry_for(n_t, L);
    out7[0] = g.L; out7[1] = g.n_tiles; out7[2] = g.lead; out7[3] = g.r; out7[4] = g.pad0;
    out7[5] = g.last_lane; out7[6] = g.last_half;
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
