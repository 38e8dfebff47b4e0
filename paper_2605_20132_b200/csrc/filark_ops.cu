// filark_ops.cu -- the two small operators beside the stream path (include/filark_ops.h):
// streaming first-order operators (running mean / de-mean / running AGC: SURVEY.md 8(f) NEXT-3,
// PAPER.md:121-122, reading R26) and display decimation (NEXT-4, reading R25).
// Both are pure streaming work: one read of the input, one write of the output.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <new>

#include "../../include/filark_ops.h"

namespace {

// ---------------------------------------------------------------------------------------------
// NEXT-3.  m[n] = alpha m[n-1] + c u[n], alpha = 1 - 1/N, c = 1/N: the same blocked scan as the
// STA/LTA averages of the stream kernel.  Channel-major: one warp per channel, a tile is 32 lanes x K
// contiguous samples; zero-state pass per lane, carry over the lanes by a 5-step shuffle scan with
// the constants alpha^(K 2^d), fix-up m[i] += alpha^(i+1) m_in.  Tiles go through shared memory both
// ways so that global accesses are coalesced (lane regions K + 1 floats apart: no bank conflicts).
constexpr int kEmaK = 16;
constexpr int kEmaWarps = 8;
struct EmaParams {
    const float* in;
    float* out;
    float* state;
    long long n_t;
    int n_ch, mode;
    float alpha, c, eps;
    float apow[kEmaK];       // alpha^(i+1)
    float aq[5];             // alpha^(K 2^d)
};

__device__ __forceinline__ float ema_out(int mode, float x, float m, float eps)
{
    return mode == FILARK_EMA_MEAN ? m : (mode == FILARK_EMA_DEMEAN ? x - m : __fdividef(x, m + eps));
}

// kVec: rows are 16-byte aligned (pointers, n_t a multiple of four): tiles move with 128-bit accesses on both
// sides of shared memory (lane regions K + 4 floats apart: 16-byte aligned and conflict-free for LDS.128);
// otherwise element by element (lane regions K + 1 floats apart).
template <bool kVec, int kMode>
__global__ void __launch_bounds__(kEmaWarps * 32) filark_ema_cm_kernel(const __grid_constant__ EmaParams p)
{
    constexpr int K = kEmaK, T = 32 * K, R = kVec ? K + 4 : K + 1;
    __shared__ __align__(16) float sm[kEmaWarps][32 * R];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* s = sm[warp];
    for (int ch = blockIdx.x * kEmaWarps + warp; ch < p.n_ch; ch += gridDim.x * kEmaWarps) {
        const float* __restrict__ row = p.in + (long long)ch * p.n_t;
        float* __restrict__ orow = p.out + (long long)ch * p.n_t;
        float carry = p.state[ch];
        for (long long t0 = 0; t0 < p.n_t; t0 += T) {
            const int n = (int)(p.n_t - t0 < T ? p.n_t - t0 : T);
            if (kVec) {
#pragma unroll
                for (int j = 0; j < K / 4; ++j) {
                    const int e = 4 * (lane + 32 * j);                       // (n is a multiple of four)
                    const float4 v = e < n ? __ldcs(reinterpret_cast<const float4*>(row + t0 + e)) : make_float4(0.f, 0.f, 0.f, 0.f);
                    *reinterpret_cast<float4*>(&s[(e / K) * R + e % K]) = v;
                }
            } else {
#pragma unroll
                for (int j = 0; j < K; ++j) {
                    const int e = lane + 32 * j;
                    s[(e / K) * R + e % K] = e < n ? row[t0 + e] : 0.0f;
                }
            }
            __syncwarp();
            float x[K], m[K];
            float acc = 0.0f;
            if (kVec) {
#pragma unroll
                for (int q = 0; q < K / 4; ++q) {
                    const float4 v = *reinterpret_cast<const float4*>(&s[lane * R + 4 * q]);
                    x[4 * q] = v.x; x[4 * q + 1] = v.y; x[4 * q + 2] = v.z; x[4 * q + 3] = v.w;
                }
            } else {
#pragma unroll
                for (int i = 0; i < K; ++i) x[i] = s[lane * R + i];
            }
#pragma unroll
            for (int i = 0; i < K; ++i) {
                const float u = kMode == FILARK_EMA_AGC ? fabsf(x[i]) : x[i];
                acc = fmaf(p.alpha, acc, p.c * u);
                m[i] = acc;
            }
            float W = acc;
            if (lane == 0) W = fmaf(p.aq[0], carry, W);
#pragma unroll
            for (int d = 0; d < 5; ++d) {
                const float U = __shfl_up_sync(0xffffffffu, W, 1 << d);
                if (lane >= (1 << d)) W = fmaf(p.aq[d], U, W);
            }
            float E = __shfl_up_sync(0xffffffffu, W, 1);
            if (lane == 0) E = carry;
            const int e_last = n - 1;
            float mlast = 0.0f;
#pragma unroll
            for (int i = 0; i < K; ++i) {
                m[i] = fmaf(p.apow[i], E, m[i]);
                if (lane * K + i == e_last) mlast = m[i];
                x[i] = ema_out(kMode, x[i], m[i], p.eps);
            }
            carry = __shfl_sync(0xffffffffu, mlast, e_last / K);
            if (kVec) {
#pragma unroll
                for (int q = 0; q < K / 4; ++q)
                    *reinterpret_cast<float4*>(&s[lane * R + 4 * q]) = make_float4(x[4 * q], x[4 * q + 1], x[4 * q + 2], x[4 * q + 3]);
                __syncwarp();
#pragma unroll
                for (int j = 0; j < K / 4; ++j) {
                    const int e = 4 * (lane + 32 * j);
                    if (e < n) __stcs(reinterpret_cast<float4*>(orow + t0 + e), *reinterpret_cast<const float4*>(&s[(e / K) * R + e % K]));
                }
            } else {
#pragma unroll
                for (int i = 0; i < K; ++i) s[lane * R + i] = x[i];
                __syncwarp();
#pragma unroll
                for (int j = 0; j < K; ++j) {
                    const int e = lane + 32 * j;
                    if (e < n) orow[t0 + e] = s[(e / K) * R + e % K];
                }
            }
            __syncwarp();
        }
        if (lane == 0) p.state[ch] = carry;
    }
}

// Time-major: a block owns 32 adjacent channels (one per lane: a warp reads 128 contiguous bytes of a time
// row) and walks the time axis in tiles of 32 x R rows; warp w is the time slice of rows [w R, (w + 1) R) of
// the tile.  The same blocked scan with the roles turned: every thread runs its R rows from rest, warp 0
// chains the 32 slices of every channel through shared memory (exact powers alpha^k for the carry, as in
// the channel-major kernel), every thread then adds alpha^(i+1) x its carry-in.  (One thread per channel
// running serially in time -- the first version -- kept 188 warps busy: 13 Gsample/s.)
constexpr int kEmaTmR = 8;
static_assert(kEmaTmR <= kEmaK, "apow[] holds alpha^1 .. alpha^K");
// kStaged: rows are 16-byte aligned (pointer, n_ch a multiple of four): the tiles arrive through a ring of
// kEmaTmStages shared-memory buffers filled by 16-byte cp.async two tiles ahead, so that about 64 KB per
// block are in flight all the time (with plain loads a block has one tile in flight during its load phase
// and nothing during the chain and the stores: 2.4 TB/s); otherwise every thread loads its own rows.
constexpr int kEmaTmStages = 3;
constexpr size_t kEmaTmStageBytes = sizeof(float) * kEmaTmStages * 32 * kEmaTmR * 32;
extern __shared__ __align__(16) float ema_stage[];
template <int kMode, bool kStaged>
__global__ void __launch_bounds__(1024, 2) filark_ema_tm_kernel(const __grid_constant__ EmaParams p)
{
    constexpr int R = kEmaTmR, T = 32 * R;
    __shared__ float sw[32][32];                 // [slice][channel]: end value from rest, then the slice's carry-in
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int n_cb = (p.n_ch + 31) / 32;
    for (int cb = blockIdx.x; cb < n_cb; cb += gridDim.x) {
        const int ch = cb * 32 + lane;
        const bool ok = ch < p.n_ch;
        float carry = (w == 0 && ok) ? p.state[ch] : 0.0f;
        // one tile = 256 rows of 128 bytes: thread (q, j) = (tid mod 8, tid / 8) copies 16 bytes of rows j and j + 128;
        // what lies outside the record or the channels is zero-filled; every call commits one group
        auto stage_tile = [&](long long t0, int stage) {
            if (t0 < p.n_t) {
                const int q = threadIdx.x & 7, j = threadIdx.x >> 3;
                const bool chok = cb * 32 + 4 * q < p.n_ch;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const long long t = t0 + j + 128 * h;
                    const unsigned dst = (unsigned)__cvta_generic_to_shared(ema_stage + (size_t)stage * T * 32 + (j + 128 * h) * 32 + 4 * q);
                    const float* src = p.in + (chok && t < p.n_t ? t * p.n_ch + cb * 32 + 4 * q : 0);
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(chok && t < p.n_t ? 16 : 0) : "memory");
                }
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        if (kStaged) {
            __syncthreads();                     // (the ring is free: the channel block before is done with it)
            for (int k = 0; k < kEmaTmStages - 1; ++k) stage_tile((long long)k * T, k);
        }
        const bool all_ch = (cb + 1) * 32 <= p.n_ch;
        const long long stride = p.n_ch;
        for (long long t0 = 0; t0 < p.n_t; t0 += T) {
            const int nt = (int)(p.n_t - t0 < T ? p.n_t - t0 : T);          // rows of this tile
            const int nv = min(max(nt - w * R, 0), R);                       // ... of this slice
            const bool full = nt == T && all_ch;                             // (block-uniform: no tests per row)
            const long long base = (t0 + (long long)w * R) * stride + ch;
            float x[R], m[R];
            if (kStaged) {
                // tile k + kEmaTmStages - 1 is asked for, tile k has landed
                const int k = (int)(t0 / T);
                stage_tile(t0 + (long long)(kEmaTmStages - 1) * T, (k + kEmaTmStages - 1) % kEmaTmStages);
                asm volatile("cp.async.wait_group %0;" ::"n"(kEmaTmStages - 1) : "memory");
                __syncthreads();
                const float* st = ema_stage + (size_t)(k % kEmaTmStages) * T * 32 + (w * R) * 32 + lane;
#pragma unroll
                for (int i = 0; i < R; ++i) x[i] = st[i * 32];
            } else {
                const float* ip = p.in + base;
#pragma unroll
                for (int i = 0; i < R; ++i) { x[i] = (full || (ok && i < nv)) ? __ldcs(ip) : 0.0f; ip += stride; }
            }
            // (rows that do not exist were zero-filled: they move nothing as long as the recurrence is not run over them)
            float acc = 0.0f;
            if (full) {
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    const float u = kMode == FILARK_EMA_AGC ? fabsf(x[i]) : x[i];
                    acc = fmaf(p.alpha, acc, p.c * u);
                    m[i] = acc;
                }
            } else {
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    const float u = kMode == FILARK_EMA_AGC ? fabsf(x[i]) : x[i];
                    if (i < nv) acc = fmaf(p.alpha, acc, p.c * u);
                    m[i] = acc;
                }
            }
            sw[w][lane] = acc;
            __syncthreads();
            if (w == 0) {
                float cin = carry;
                if (nt == T) {
                    const float aR = p.apow[R - 1];
#pragma unroll 8
                    for (int s = 0; s < 32; ++s) {
                        const float end = sw[s][lane];
                        sw[s][lane] = cin;
                        cin = fmaf(aR, cin, end);
                    }
                } else {
#pragma unroll 4
                    for (int s = 0; s < 32; ++s) {
                        const int nvs = min(max(nt - s * R, 0), R);
                        const float end = sw[s][lane];
                        sw[s][lane] = cin;
                        if (nvs > 0) cin = fmaf(p.apow[nvs - 1], cin, end);
                    }
                }
                carry = cin;
            }
            __syncthreads();
            const float E = sw[w][lane];
            float* op = p.out + base;
            if (full) {
#pragma unroll
                for (int i = 0; i < R; ++i) { __stcs(op, ema_out(kMode, x[i], fmaf(p.apow[i], E, m[i]), p.eps)); op += stride; }
            } else {
#pragma unroll
                for (int i = 0; i < R; ++i) {
                    if (ok && i < nv) __stcs(op, ema_out(kMode, x[i], fmaf(p.apow[i], E, m[i]), p.eps));
                    op += stride;
                }
            }
            __syncthreads();
        }
        if (w == 0 && ok) p.state[ch] = carry;
    }
}

// ---------------------------------------------------------------------------------------------
// NEXT-4.  Column j of a channel covers input samples [a_j, a_{j+1}), a_j = floor(j n_t / width).
struct DecParams {
    const float* in;
    float* out;
    long long n_t, pitch;
    int n_ch, width, mode;
    int slice;               // channel-major peak mode: samples a warp can stage (0: column by column)
};
__device__ __forceinline__ long long col_start(long long j, long long n_t, int width) { return j * n_t / width; }

__device__ __forceinline__ float lin_at(const float* row, long long stride, long long n_t, int j, int width)
{
    const double pos = width > 1 ? (double)j * (double)(n_t - 1) / (double)(width - 1) : 0.0;
    long long i = (long long)pos;
    if (i > n_t - 1) i = n_t - 1;
    const float f = (float)(pos - (double)i);
    const float x0 = row[i * stride], x1 = row[(i + 1 < n_t ? i + 1 : i) * stride];
    return fmaf(x1 - x0, f, x0);
}

// Channel-major: grid (column groups, channels).  Narrow columns (<= 32 samples): one thread per column
// (a warp reads 32 adjacent columns: one contiguous stretch of the row).  Wide columns, peak mode: a warp
// takes 32 adjacent columns at a time, copies their stretch of the row into its slice of shared memory with
// coalesced loads (one read of every sample) and every lane then walks its own column there; stretches
// longer than the slice (columns of more than 64 samples) go column by column, the lanes striding through a
// column and the largest magnitude -- the first one on ties -- found by a shuffle reduction on
// (magnitude, position).
constexpr int kDecSlice = 2048;                                   // samples of a warp's slice
// (a launch asks for the slice its columns need: 32 columns of ceil(n_t / width) samples, at most kDecSlice)
__device__ __forceinline__ int dec_at(int i) { return i + (i >> 5); }   // (one pad per 32: the lanes' columns start in different banks)

__global__ void __launch_bounds__(128) filark_decimate_cm_kernel(const __grid_constant__ DecParams p)
{
    extern __shared__ float dec_slices[];            // wide columns in peak mode only: 4 slices (kDecSmemBytes)
    const int ch = blockIdx.y;
    const float* __restrict__ row = p.in + (long long)ch * p.pitch;
    float* __restrict__ orow = p.out + (long long)ch * p.width;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool narrow = p.n_t <= 32LL * p.width;
    if (p.mode != FILARK_DECIMATE_PEAK || narrow) {
        const int j = blockIdx.x * blockDim.x + threadIdx.x;
        if (j >= p.width) return;
        const long long a = col_start(j, p.n_t, p.width);
        float v;
        if (p.mode == FILARK_DECIMATE_DROP) {
            v = row[a];
        } else if (p.mode == FILARK_DECIMATE_LINEAR) {
            v = lin_at(row, 1, p.n_t, j, p.width);
        } else {
            long long b = col_start(j + 1, p.n_t, p.width);
            if (b <= a) b = a + 1;
            v = row[a];
            float best = fabsf(v);
            for (long long n = a + 1; n < b; ++n) {
                const float s = row[n];
                if (fabsf(s) > best) { best = fabsf(s); v = s; }
            }
        }
        orow[j] = v;
        return;
    }
    float* s = dec_slices + warp * (p.slice + p.slice / 32 + 1);
    for (int j0 = (blockIdx.x * 4 + warp) * 32; j0 < p.width; j0 += gridDim.x * 4 * 32) {
        const int j1 = min(p.width, j0 + 32);
        const long long a0 = col_start(j0, p.n_t, p.width), a1 = col_start(j1, p.n_t, p.width);
        if (a1 - a0 <= p.slice) {
            const int len = (int)(a1 - a0);
            // (eight loads in flight per lane: the copy is the part that waits for memory)
            for (int i0 = lane; i0 < len; i0 += 256) {
                float v[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) v[u] = i0 + 32 * u < len ? __ldcs(row + a0 + i0 + 32 * u) : 0.0f;
#pragma unroll
                for (int u = 0; u < 8; ++u) if (i0 + 32 * u < len) s[dec_at(i0 + 32 * u)] = v[u];
            }
            __syncwarp();
            const int j = j0 + lane;
            if (j < j1) {
                const int a = (int)(col_start(j, p.n_t, p.width) - a0), b = (int)(col_start(j + 1, p.n_t, p.width) - a0);
                float v = s[dec_at(a)], best = fabsf(v);
                int n = a + 1;
                for (; n + 4 <= b; n += 4) {                  // (four loads in flight; the comparisons stay in time order)
                    const float x0 = s[dec_at(n)], x1 = s[dec_at(n + 1)], x2 = s[dec_at(n + 2)], x3 = s[dec_at(n + 3)];
                    if (fabsf(x0) > best) { best = fabsf(x0); v = x0; }
                    if (fabsf(x1) > best) { best = fabsf(x1); v = x1; }
                    if (fabsf(x2) > best) { best = fabsf(x2); v = x2; }
                    if (fabsf(x3) > best) { best = fabsf(x3); v = x3; }
                }
                for (; n < b; ++n) {
                    const float x = s[dec_at(n)];
                    if (fabsf(x) > best) { best = fabsf(x); v = x; }
                }
                orow[j] = v;
            }
            __syncwarp();
            continue;
        }
        for (int j = j0; j < j1; ++j) {
            const long long a = col_start(j, p.n_t, p.width), b = col_start(j + 1, p.n_t, p.width);
            float v = 0.0f, best = -1.0f;
            long long at = b;
            for (long long n = a + lane; n < b; n += 32) {
                const float x = row[n];
                if (fabsf(x) > best) { best = fabsf(x); v = x; at = n; }
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                const float ob = __shfl_xor_sync(0xffffffffu, best, d), ov = __shfl_xor_sync(0xffffffffu, v, d);
                const long long oa = __shfl_xor_sync(0xffffffffu, at, d);
                if (ob > best || (ob == best && oa < at)) { best = ob; v = ov; at = oa; }
            }
            if (lane == 0) orow[j] = v;
        }
    }
}

// Time-major: adjacent threads are adjacent channels; a thread walks the samples of its columns in time.
__global__ void __launch_bounds__(128) filark_decimate_tm_kernel(const __grid_constant__ DecParams p, int cols_per_block)
{
    const int ch = blockIdx.x * blockDim.x + threadIdx.x;
    if (ch >= p.n_ch) return;
    const float* __restrict__ col = p.in + ch;
    const int j0 = blockIdx.y * cols_per_block, j1 = min(p.width, j0 + cols_per_block);
    for (int j = j0; j < j1; ++j) {
        const long long a = col_start(j, p.n_t, p.width);
        float v;
        if (p.mode == FILARK_DECIMATE_DROP) {
            v = col[a * p.pitch];
        } else if (p.mode == FILARK_DECIMATE_LINEAR) {
            v = lin_at(col, p.pitch, p.n_t, j, p.width);
        } else {
            long long b = col_start(j + 1, p.n_t, p.width);
            if (b <= a) b = a + 1;
            v = col[a * p.pitch];
            float best = fabsf(v);
            for (long long n = a + 1; n < b; ++n) {
                const float s = col[n * p.pitch];
                if (fabsf(s) > best) { best = fabsf(s); v = s; }
            }
        }
        p.out[(long long)j * p.n_ch + ch] = v;
    }
}

}  // namespace

// cudaFuncAttributeMaxDynamicSharedMemorySize is per device: set it on every launch of a staged kernel (a
// cheap host call; the streaming operators are not launch-rate bound).
static cudaError_t ema_smem_attr_once(int, const void* func, size_t bytes)
{
    return cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

struct filark_ema {
    int device, n_ch, n_len, mode, layout;
    float eps;
    EmaParams proto;
    float* d_state;
    int n_sm;
};

extern "C" {

filark_status_t filark_ema_create(filark_ema_t** out, int n_ch, int n_len, int mode, float eps, int layout)
{
    if (!out || n_ch <= 0 || n_len < 1 || mode < FILARK_EMA_MEAN || mode > FILARK_EMA_AGC || !(eps >= 0.0f) ||
        !std::isfinite(eps) || (layout != FILARK_LAYOUT_CHANNEL_MAJOR && layout != FILARK_LAYOUT_TIME_MAJOR))
        return FILARK_ERR_INVALID_ARG;
    filark_ema* h = new (std::nothrow) filark_ema();
    if (!h) return FILARK_ERR_ALLOC;
    h->n_ch = n_ch; h->n_len = n_len; h->mode = mode; h->layout = layout; h->eps = eps;
    cudaError_t e = cudaGetDevice(&h->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device);
    if (e == cudaSuccess) e = cudaMalloc((void**)&h->d_state, sizeof(float) * (size_t)n_ch);
    if (e == cudaSuccess) e = cudaMemset(h->d_state, 0, sizeof(float) * (size_t)n_ch);
    if (e != cudaSuccess) {
        const bool oom = e == cudaErrorMemoryAllocation;
        cudaFree(h->d_state); delete h; cudaGetLastError();
        return oom ? FILARK_ERR_ALLOC : FILARK_ERR_CUDA;
    }
    // constants in float64, rounded last: alpha^k = exp(k log1p(-1/N))
    EmaParams& p = h->proto;
    p = EmaParams{};
    const double c = 1.0 / (double)n_len;
    const double la = n_len > 1 ? std::log1p(-c) : -INFINITY;          // N = 1: alpha = 0
    auto apow = [&](double k) { return n_len > 1 ? std::exp(k * la) : 0.0; };
    p.n_ch = n_ch; p.mode = mode; p.eps = eps; p.alpha = (float)(1.0 - c); p.c = (float)c; p.state = h->d_state;
    for (int i = 0; i < kEmaK; ++i) p.apow[i] = (float)apow(i + 1.0);
    for (int d = 0; d < 5; ++d) p.aq[d] = (float)apow((double)kEmaK * (double)(1 << d));
    *out = h;
    return FILARK_OK;
}

filark_status_t filark_ema_push(filark_ema_t* h, const float* d_in, long long n_t, float* d_out, cudaStream_t stream)
{
    if (!h || n_t < 0) return FILARK_ERR_INVALID_ARG;
    if (n_t == 0) return FILARK_OK;
    if (!d_in || !d_out || n_t > 0x7fff0000LL) return FILARK_ERR_INVALID_ARG;
    if (((uintptr_t)d_in | (uintptr_t)d_out) & 3u) return FILARK_ERR_ALIGNMENT;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return FILARK_ERR_CUDA;
    if (dev != h->device) return FILARK_ERR_DEVICE_MISMATCH;
    EmaParams p = h->proto;
    p.in = d_in; p.out = d_out; p.n_t = n_t;
    if (h->layout == FILARK_LAYOUT_CHANNEL_MAJOR) {
        int grid = (h->n_ch + kEmaWarps - 1) / kEmaWarps;
        const int cap = h->n_sm * 3;                 // (measured: more rows in flight at once cost DRAM efficiency, 4.6 vs 5.7 TB/s)
        if (grid > cap) grid = cap;
        // (d_out == d_in is allowed: a tile is read completely before it is written)
        const bool vec = (((uintptr_t)d_in | (uintptr_t)d_out) & 15u) == 0 && (n_t & 3) == 0;
#define FK_EMA_LAUNCH(V, M) filark_ema_cm_kernel<V, M><<<grid, kEmaWarps * 32, 0, stream>>>(p)
        if (vec) {
            if (h->mode == FILARK_EMA_MEAN) FK_EMA_LAUNCH(true, FILARK_EMA_MEAN);
            else if (h->mode == FILARK_EMA_DEMEAN) FK_EMA_LAUNCH(true, FILARK_EMA_DEMEAN);
            else FK_EMA_LAUNCH(true, FILARK_EMA_AGC);
        } else {
            if (h->mode == FILARK_EMA_MEAN) FK_EMA_LAUNCH(false, FILARK_EMA_MEAN);
            else if (h->mode == FILARK_EMA_DEMEAN) FK_EMA_LAUNCH(false, FILARK_EMA_DEMEAN);
            else FK_EMA_LAUNCH(false, FILARK_EMA_AGC);
        }
#undef FK_EMA_LAUNCH
    } else {
        int grid = (h->n_ch + 31) / 32;
        if (grid > 2 * h->n_sm) grid = 2 * h->n_sm;
        const bool staged = ((uintptr_t)d_in & 15u) == 0 && (h->n_ch & 3) == 0;
        cudaError_t e = cudaSuccess;
#define FK_EMA_TM(M)                                                                                              \
        if (staged) {                                                                                             \
            e = ema_smem_attr_once(h->device, (const void*)filark_ema_tm_kernel<M, true>, kEmaTmStageBytes);      \
            if (e == cudaSuccess) filark_ema_tm_kernel<M, true><<<grid, 1024, kEmaTmStageBytes, stream>>>(p);     \
        } else {                                                                                                  \
            filark_ema_tm_kernel<M, false><<<grid, 1024, 0, stream>>>(p);                                         \
        }
        if (h->mode == FILARK_EMA_MEAN) { FK_EMA_TM(FILARK_EMA_MEAN) }
        else if (h->mode == FILARK_EMA_DEMEAN) { FK_EMA_TM(FILARK_EMA_DEMEAN) }
        else { FK_EMA_TM(FILARK_EMA_AGC) }
#undef FK_EMA_TM
        if (e != cudaSuccess) return FILARK_ERR_CUDA;
    }
    return cudaGetLastError() == cudaSuccess ? FILARK_OK : FILARK_ERR_CUDA;
}

filark_status_t filark_ema_reset(filark_ema_t* h, cudaStream_t stream)
{
    if (!h) return FILARK_ERR_INVALID_ARG;
    return cudaMemsetAsync(h->d_state, 0, sizeof(float) * (size_t)h->n_ch, stream) == cudaSuccess ? FILARK_OK : FILARK_ERR_CUDA;
}

filark_status_t filark_ema_destroy(filark_ema_t* h)
{
    if (!h) return FILARK_OK;
    int cur = -1;
    const bool have_cur = cudaGetDevice(&cur) == cudaSuccess;
    const bool switched = have_cur && cur != h->device && cudaSetDevice(h->device) == cudaSuccess;
    cudaDeviceSynchronize();
    cudaFree(h->d_state);
    if (switched) cudaSetDevice(cur);
    cudaGetLastError();
    delete h;
    return FILARK_OK;
}

filark_status_t filark_decimate(const float* d_in, int n_ch, long long n_t, long long pitch, int layout, int mode,
                                int width, float* d_out, cudaStream_t stream)
{
    if (!d_in || !d_out || n_ch <= 0 || n_t <= 0 || width <= 0 || n_t > 0x7fff0000LL) return FILARK_ERR_INVALID_ARG;
    if (mode < FILARK_DECIMATE_DROP || mode > FILARK_DECIMATE_LINEAR) return FILARK_ERR_INVALID_ARG;
    const bool cm = layout == FILARK_LAYOUT_CHANNEL_MAJOR;
    if (!cm && layout != FILARK_LAYOUT_TIME_MAJOR) return FILARK_ERR_INVALID_ARG;
    if (pitch < (cm ? n_t : (long long)n_ch)) return FILARK_ERR_INVALID_ARG;
    if (((uintptr_t)d_in | (uintptr_t)d_out) & 3u) return FILARK_ERR_ALIGNMENT;
    const uintptr_t a0 = (uintptr_t)d_in, a1 = a0 + sizeof(float) * (size_t)(((cm ? n_ch : n_t) - 1) * pitch + (cm ? n_t : n_ch));
    const uintptr_t b0 = (uintptr_t)d_out, b1 = b0 + sizeof(float) * (size_t)n_ch * (size_t)width;
    if (a0 < b1 && b0 < a1) return FILARK_ERR_INVALID_ARG;
    DecParams p{d_in, d_out, n_t, pitch, n_ch, width, mode, 0};
    if (cm) {
        if (n_ch > 65535) return FILARK_ERR_INVALID_ARG;
        const bool per_thread = mode != FILARK_DECIMATE_PEAK || n_t <= 32LL * width;
        int gx = (width + 127) / 128;                 // 128 columns per block either way (wide: 32 per warp)
        if (!per_thread && gx > 64) gx = 64;
        size_t smem = 0;
        if (!per_thread) {
            const long long need = 32 * ((n_t + width - 1) / width) + 32;
            p.slice = need <= kDecSlice ? (int)need : 0;      // wider columns: column by column, no staging
            smem = sizeof(float) * 4 * (size_t)(p.slice + p.slice / 32 + 1);
        }
        filark_decimate_cm_kernel<<<dim3((unsigned)gx, (unsigned)n_ch), 128, smem, stream>>>(p);
    } else {
        int gy = (width + 31) / 32;
        if (gy > 65535) gy = 65535;
        const int cols = (width + gy - 1) / gy;
        filark_decimate_tm_kernel<<<dim3((unsigned)((n_ch + 127) / 128), (unsigned)gy), 128, 0, stream>>>(p, cols);
    }
    return cudaGetLastError() == cudaSuccess ? FILARK_OK : FILARK_ERR_CUDA;
}

}  // extern "C"
