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

struct filark_stream {
    int device;
    int n_ch, n_sec, sta_len, lta_len, layout;
    unsigned flags;
    Section sec[kMaxSec];
    double gain;
    float* d_tab;
    float* d_state;
    Counter* d_ctr;
    size_t tab_floats, state_floats;
    int last_cuda_error;
    long long launches, samples;
    long long cached_tail_rem;      // n_t % kTile the cached TailTab was built for (-1: none)
    TailTab tail;
    int tail_len, tail_nfull, tail_part, tail_jl, tail_magic;
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

// Static table for full tiles (layout documented in filark_kernels.cuh).
static void build_static_table(const filark_stream* h, float* tab)
{
    std::memset(tab, 0, sizeof(float) * h->tab_floats);
    for (int k = 0; k < h->n_sec; ++k) {
        const Section& s = h->sec[k];
        float* T = tab + k * kSecStride;
        const int kind = s.kind == KIND_R ? kKindR : kKindT;
        std::memcpy(&T[0], &kind, sizeof(int));
        for (int i = 0; i < 5; ++i) T[kOffCoef + i] = (float)s.coef[i];
        Mat2 P[kSteps];
        scan_powers(s, kL, P);
        for (int d = 0; d < kSteps; ++d) put_mat(T + kOffP + 4 * d, P[d]);
        double g[2 * kL];
        fixup_rows(s, kL, g);
        for (int i = 0; i < 2 * kL; ++i) T[kOffG + i] = (float)g[i];
    }
    float* AV = tab + h->n_sec * kSecStride;
    const double cs = 1.0 / h->sta_len, cl = 1.0 / h->lta_len;
    const double as = 1.0 - cs, al = 1.0 - cl;
    AV[0] = (float)as; AV[1] = (float)al; AV[2] = (float)cs; AV[3] = (float)cl;
    for (int d = 0; d < kSteps; ++d) {
        const double e = (double)kL * (double)(1 << d);
        AV[4 + d] = (float)(-std::expm1(e * std::log1p(-cs)));   // 1 - as^e without cancellation
        AV[9 + d] = (float)(-std::expm1(e * std::log1p(-cl)));
    }
}

static double one_minus_pow(double c, double e)      // 1 - (1-c)^e, accurate for tiny c
{
    if (c >= 1.0) return e > 0 ? 1.0 : 0.0;
    return -std::expm1(e * std::log1p(-c));
}

// Geometry + table of the ragged tail tile for rem = n_t % kTile samples (rem >= 1).
static void build_tail(filark_stream* h, int rem)
{
    if (h->cached_tail_rem == rem) return;
    const int len = (rem + 31) / 32;
    const int nfull = rem / len, part = rem % len;
    h->tail_len = len; h->tail_nfull = nfull; h->tail_part = part;
    h->tail_jl = part > 0 ? nfull : nfull - 1;
    h->tail_magic = (65536 + len - 1) / len;
    const int end_len = part > 0 ? part : len;
    std::memset(&h->tail, 0, sizeof(TailTab));
    for (int k = 0; k < h->n_sec; ++k) {
        Mat2 P[kSteps];
        scan_powers(h->sec[k], len, P);
        for (int d = 0; d < kSteps; ++d) put_mat(&h->tail.P[k][d][0], P[d]);
        put_mat(&h->tail.Aend[k][0], mpow(h->sec[k].A, end_len));
    }
    const double cs = 1.0 / h->sta_len, cl = 1.0 / h->lta_len;
    for (int d = 0; d < kSteps; ++d) {
        h->tail.beta_s[d] = (float)one_minus_pow(cs, (double)len * (1 << d));
        h->tail.beta_l[d] = (float)one_minus_pow(cl, (double)len * (1 << d));
    }
    h->tail.beta_end_s = (float)one_minus_pow(cs, end_len);
    h->tail.beta_end_l = (float)one_minus_pow(cl, end_len);
    h->cached_tail_rem = rem;
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
    if (flags & ~FILARK_FLAG_SERIAL_SCAN) return FILARK_ERR_INVALID_ARG;
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
    h->layout = layout; h->flags = flags; h->cached_tail_rem = -1;
    h->tab_floats = (size_t)n_sec * kSecStride + kAvgFloats;
    h->state_floats = (size_t)n_ch * (size_t)(2 * n_sec + 2);
    cudaError_t e = cudaGetDevice(&h->device);
    float* tab = nullptr;
    if (e == cudaSuccess) {
        tab = (float*)std::malloc(sizeof(float) * h->tab_floats);
        if (!tab) { delete h; return FILARK_ERR_ALLOC; }
        build_static_table(h, tab);
    }
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_tab, sizeof(float) * h->tab_floats);
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_state, sizeof(float) * h->state_floats);
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_ctr, sizeof(Counter));
    if (e == cudaSuccess) e = cudaMemcpy(h->d_tab, tab, sizeof(float) * h->tab_floats, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(h->d_state, 0, sizeof(float) * h->state_floats);
    if (e == cudaSuccess) e = cudaMemset(h->d_ctr, 0, sizeof(Counter));
    std::free(tab);
    if (e != cudaSuccess) {
        const bool oom = e == cudaErrorMemoryAllocation;
        cudaFree(h->d_tab); cudaFree(h->d_state); cudaFree(h->d_ctr);
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
    cudaFree(h->d_tab); cudaFree(h->d_state); cudaFree(h->d_ctr);
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
    if (e == cudaSuccess) e = cudaMemsetAsync(h->d_ctr, 0, sizeof(Counter), stream);
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
    p.tab = h->d_tab; p.state = h->d_state; p.ctr = h->d_ctr;
    p.n_t = n_t; p.in_pitch = in_pitch; p.out_pitch = out_pitch;
    p.n_ch = h->n_ch; p.n_sec = h->n_sec;
    p.lta_len = h->lta_len;
    p.gain = (float)h->gain;
    p.ratio = (float)((double)h->lta_len / (double)h->sta_len);
    p.lta_thr = (float)(1e-30 * (double)h->lta_len);      // lta <= 1e-30  <=>  lta~ <= 1e-30 N_l
    const size_t tab_bytes = sizeof(float) * ((h->tab_floats + 3) & ~(size_t)3);
    const int ns = 2 * h->n_sec + 2;

    if ((h->flags & FILARK_FLAG_SERIAL_SCAN) || !cm) {
        // Serial diagnostic kernel; also the time-major path until the blocked time-major
        // kernel lands.
        const long long sc_in = cm ? in_pitch : 1, st_in = cm ? 1 : in_pitch;
        const long long sc_out = cm ? out_pitch : 1, st_out = cm ? 1 : out_pitch;
        const long long state_sc = cm ? ns : 1, state_sk = cm ? 1 : h->n_ch;
        const int block = 128, grid = (h->n_ch + block - 1) / block;
        filark_push_serial_kernel<<<grid, block, tab_bytes, stream>>>(p, sc_in, st_in, sc_out, st_out,
                                                                      state_sc, state_sk);
    } else {
        p.n_full = (int)(n_t / kTile);
        const int rem = (int)(n_t % kTile);
        if (rem > 0) {
            build_tail(h, rem);
            p.tail_len = h->tail_len; p.tail_nfull = h->tail_nfull; p.tail_part = h->tail_part;
            p.tail_jl = h->tail_jl; p.tail_magic = h->tail_magic;
        }
        const uintptr_t all = (uintptr_t)d_in | (uintptr_t)d_filt | (uintptr_t)d_cf;
        p.vec4 = ((all & 15u) == 0 && (in_pitch & 3) == 0 && (out_pitch & 3) == 0) ? 1 : 0;
        const int st_floats = (ns + 3) & ~3;
        const size_t smem = tab_bytes + sizeof(float) * (size_t)kWarps * (32 * kPitch + st_floats);
        const int grid = (h->n_ch + kWarps - 1) / kWarps;
        filark_push_cm_kernel<<<grid, kWarps * 32, smem, stream>>>(p, h->tail);
    }
    e = cudaGetLastError();
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

int filark_debug_tail_geometry(long long n_t, int* n_full, int* len, int* nfull, int* part, int* jl)
{
    if (n_t < 0) return (int)FILARK_ERR_INVALID_ARG;
    const int rem = (int)(n_t % kTile);
    if (n_full) *n_full = (int)(n_t / kTile);
    int l = 0, nf = 0, pt = 0, j = -1;
    if (rem > 0) { l = (rem + 31) / 32; nf = rem / l; pt = rem % l; j = pt > 0 ? nf : nf - 1; }
    if (len) *len = l;
    if (nfull) *nfull = nf;
    if (part) *part = pt;
    if (jl) *jl = j;
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
