// filark_kernels.cuh -- sm_100a kernels of the fused SOS + STA/LTA stream path.
//
// Steps (include/filark_stream.h): S0 load, S1 per-section local scan,
// S2 warp-shuffle combine, S3 fix-up + carried state, S4 energy, S5 STA/LTA scans,
// S6 ratio + warm-up, S7 store.  One launch per push; the chunk is read once from HBM and
// each output is written once.
//
// Channel-major mapping (time contiguous): one warp owns one channel.  A tile is 32 lanes x
// len consecutive samples (len = 32 in a full tile, 1..32 in the ragged tail tile of a push);
// a lane's samples stay in registers through every section and the STA/LTA.  Tiles of a
// channel are processed in time order by the same warp; the carried state sits in shared
// memory between tiles and in global memory between pushes.  Coalesced float4 global accesses
// are transposed through a padded per-warp shared tile ([32][36] floats, conflict-free both
// ways).
//
// The recurrences are exact restatements of the oracle's definition:
//   section:  s[n] = A s[n-1] + B x[n],  y[n] = C s[n-1] + D x[n]           (design.hpp)
//   sub-block with carry-in s_in, local pass from zero state giving y_loc, v:
//             y[i] = y_loc[i] + (C A^i) s_in,   s_out = A^len s_in + v
//   averages: m~[n] = alpha m~[n-1] + e[n]  (m~ = m * N),  cf = (N_l/N_s) s~/l~
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace filark {

constexpr int kL = 32;                 // samples per lane in a full tile
constexpr int kTile = 32 * kL;         // samples per full tile
constexpr int kPitch = 36;             // floats per sub-block row of the transpose tile
constexpr int kWarps = 4;              // warps (= channels in flight) per CTA
constexpr int kMaxSec = 16;
constexpr int kSteps = 5;              // log2(32) scan steps
constexpr int kKindT = 0, kKindR = 1;

// ---- static (per handle) device table, floats ------------------------------------------------
// per section, stride kSecStride:
//   [0]      kind (int bits)
//   [1..5]   local-pass coefficients (kind R: sigma omega c1 c2 | kind T: b0 b1 b2 -a1 -a2)
//   [8..27]  P[d] = A^(32 2^d), d = 0..4, row-major 2x2
//   [32..95] fix-up rows g[i] = C A^i, i < 32, interleaved (g1, g2)
constexpr int kSecStride = 96;
constexpr int kOffCoef = 1;
constexpr int kOffP = 8;
constexpr int kOffG = 32;
// after the sections, the averages block:
//   [0] alpha_s [1] alpha_l [2] c_s = 1/N_s [3] c_l = 1/N_l
//   [4..8] beta_s[d] = 1 - alpha_s^(32 2^d)   [9..13] beta_l[d]
constexpr int kAvgFloats = 16;

// ---- per-push table for the ragged tail tile (kernel parameter space) -------------------------
struct __align__(16) TailTab {
    float P[kMaxSec][kSteps][4];       // A^(len 2^d)
    float Aend[kMaxSec][4];            // A^part (or A^len when no lane is partial)
    float beta_s[kSteps], beta_l[kSteps];
    float beta_end_s, beta_end_l;
};

struct Counter { unsigned long long g; unsigned int ticket; unsigned int pad; };

struct PushParams {
    const float* in;
    float* filt;
    float* cf;
    const float* tab;        // static table (device)
    float* state;            // channel-major: [n_ch][2 n_sec + 2]; time-major: [2 n_sec + 2][n_ch]
    Counter* ctr;
    long long n_t, in_pitch, out_pitch;
    int n_ch, n_sec;
    int n_full;              // full tiles per channel
    int tail_len;            // sub-block length of the tail tile (0: none)
    int tail_nfull;          // lanes holding tail_len samples
    int tail_part;           // samples in the partial lane (0: none)
    int tail_jl;             // lane whose end state is the carry-out
    int tail_magic;          // ceil(65536 / tail_len): e / tail_len == (e * magic) >> 16, e < 1024
    int lta_len;
    int vec4;                // float4 global accesses are legal (alignment + pitch)
    float gain, ratio, lta_thr;
};

__device__ __forceinline__ float ld_stream(const float* p) { return __ldcs(p); }
__device__ __forceinline__ float4 ld_stream4(const float* p) { return __ldcs(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ void st_stream(float* p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream4(float* p, float4 v) { __stcs(reinterpret_cast<float4*>(p), v); }

// S0: bring the tile's samples of one channel into registers, lane j <- [j len, (j+1) len).
template <bool GEN>
__device__ __forceinline__ void stage_in(float (&x)[kL], const float* __restrict__ src, float* buf,
                                         int lane, bool vec4, int len, int n_valid, int magic,
                                         float gain)
{
    if (!GEN) {
        if (vec4) {
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const float4 v = ld_stream4(src + 128 * m + 4 * lane);
                *reinterpret_cast<float4*>(buf + (4 * m + (lane >> 3)) * kPitch + 4 * (lane & 7)) = v;
            }
        } else {
#pragma unroll
            for (int m = 0; m < 32; ++m) buf[m * kPitch + lane] = ld_stream(src + 32 * m + lane);
        }
    } else {
        for (int m = 0; m < len; ++m) {
            const int e = 32 * m + lane;
            const int row = (e * magic) >> 16, col = e - row * len;
            buf[row * kPitch + col] = e < n_valid ? ld_stream(src + e) : 0.0f;
        }
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (GEN && 4 * q >= len) break;
        const float4 v = *reinterpret_cast<const float4*>(buf + lane * kPitch + 4 * q);
        x[4 * q + 0] = v.x * gain; x[4 * q + 1] = v.y * gain;
        x[4 * q + 2] = v.z * gain; x[4 * q + 3] = v.w * gain;
    }
    __syncwarp();
}

// S7: registers -> one output array, same geometry as stage_in.
template <bool GEN>
__device__ __forceinline__ void stage_out(const float (&x)[kL], float* __restrict__ dst, float* buf,
                                          int lane, bool vec4, int len, int n_valid, int magic)
{
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        if (GEN && 4 * q >= len) break;
        *reinterpret_cast<float4*>(buf + lane * kPitch + 4 * q) =
            make_float4(x[4 * q], x[4 * q + 1], x[4 * q + 2], x[4 * q + 3]);
    }
    __syncwarp();
    if (!GEN) {
        if (vec4) {
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const float4 v = *reinterpret_cast<const float4*>(
                    buf + (4 * m + (lane >> 3)) * kPitch + 4 * (lane & 7));
                st_stream4(dst + 128 * m + 4 * lane, v);
            }
        } else {
#pragma unroll
            for (int m = 0; m < 32; ++m) st_stream(dst + 32 * m + lane, buf[m * kPitch + lane]);
        }
    } else {
        for (int m = 0; m < len; ++m) {
            const int e = 32 * m + lane;
            const int row = (e * magic) >> 16, col = e - row * len;
            if (e < n_valid) st_stream(dst + e, buf[row * kPitch + col]);
        }
    }
    __syncwarp();
}

// S2: inclusive scan over lanes of v_j <- v_j + P^(2^d) v_(j-2^d) with constant 2x2 blocks.
__device__ __forceinline__ void scan2(float& v1, float& v2, const float* __restrict__ P, int lane)
{
#pragma unroll
    for (int d = 0; d < kSteps; ++d) {
        const float4 m = reinterpret_cast<const float4*>(P)[d];
        const float u1 = __shfl_up_sync(0xffffffffu, v1, 1 << d);
        const float u2 = __shfl_up_sync(0xffffffffu, v2, 1 << d);
        if (lane >= (1 << d)) {
            v1 = fmaf(m.x, u1, fmaf(m.y, u2, v1));
            v2 = fmaf(m.z, u1, fmaf(m.w, u2, v2));
        }
    }
}

// 1-D version for the averages, in the form v += u - beta u (beta = 1 - alpha^(len 2^d)), which
// keeps the unit DC gain of the average to fp32 relative accuracy (reading R13).
__device__ __forceinline__ void scan1(float& v, const float* __restrict__ beta, int lane)
{
#pragma unroll
    for (int d = 0; d < kSteps; ++d) {
        const float u = __shfl_up_sync(0xffffffffu, v, 1 << d);
        if (lane >= (1 << d)) v += fmaf(-beta[d], u, u);
    }
}

// One tile of one channel: S0..S7.
template <bool GEN>
__device__ __forceinline__ void process_tile(const PushParams& p, const TailTab& tt,
                                             const float* __restrict__ stab, float* buf, float* wst,
                                             int ch, long long t0, int lane, unsigned long long g0)
{
    const int len = GEN ? p.tail_len : kL;
    const int n_valid = GEN ? p.tail_nfull * len + p.tail_part : kTile;
    const int mylen = !GEN ? kL : (lane < p.tail_nfull ? len : (lane == p.tail_nfull ? p.tail_part : 0));
    const int jl = GEN ? p.tail_jl : 31;
    const bool vec4 = p.vec4 != 0;
    float x[kL];

    stage_in<GEN>(x, p.in + (long long)ch * p.in_pitch + t0, buf, lane, vec4, len, n_valid,
                  p.tail_magic, p.gain);

    // ---- S1..S3 per section -------------------------------------------------------------------
    for (int k = 0; k < p.n_sec; ++k) {
        const float* __restrict__ T = stab + k * kSecStride;
        const int kind = __float_as_int(T[0]);
        float v1 = 0.0f, v2 = 0.0f;
        if (kind == kKindR) {
            const float sg = T[kOffCoef + 0], om = T[kOffCoef + 1];
            const float c1 = T[kOffCoef + 2], c2 = T[kOffCoef + 3];
#pragma unroll
            for (int i = 0; i < kL; ++i) {
                if (GEN && i >= len) break;
                const float xi = x[i];
                const float y = fmaf(c1, v1, fmaf(c2, v2, xi));
                const float n1 = fmaf(sg, v1, fmaf(om, v2, xi));
                const float n2 = fmaf(sg, v2, -om * v1);
                if (!GEN || i < mylen) { v1 = n1; v2 = n2; }
                x[i] = y;
            }
        } else {
            const float b0 = T[kOffCoef + 0], b1 = T[kOffCoef + 1], b2 = T[kOffCoef + 2];
            const float na1 = T[kOffCoef + 3], na2 = T[kOffCoef + 4];
#pragma unroll
            for (int i = 0; i < kL; ++i) {
                if (GEN && i >= len) break;
                const float xi = x[i];
                const float y = fmaf(b0, xi, v1);
                const float n1 = fmaf(na1, y, fmaf(b1, xi, v2));
                const float n2 = fmaf(na2, y, b2 * xi);
                if (!GEN || i < mylen) { v1 = n1; v2 = n2; }
                x[i] = y;
            }
        }
        // carried state of this section (true state before the tile's first sample)
        const float S1 = wst[2 * k], S2 = wst[2 * k + 1];
        const float* __restrict__ P = GEN ? &tt.P[k][0][0] : T + kOffP;
        float w1 = v1, w2 = v2;
        if (lane == 0) {
            w1 = fmaf(P[0], S1, fmaf(P[1], S2, w1));
            w2 = fmaf(P[2], S1, fmaf(P[3], S2, w2));
        }
        scan2(w1, w2, P, lane);
        float a = __shfl_up_sync(0xffffffffu, w1, 1);
        float b = __shfl_up_sync(0xffffffffu, w2, 1);
        if (lane == 0) { a = S1; b = S2; }
        float o1, o2;
        if (!GEN) {
            o1 = w1; o2 = w2;
        } else {
            const float* __restrict__ E = &tt.Aend[k][0];
            o1 = fmaf(E[0], a, fmaf(E[1], b, v1));
            o2 = fmaf(E[2], a, fmaf(E[3], b, v2));
        }
        o1 = __shfl_sync(0xffffffffu, o1, jl);
        o2 = __shfl_sync(0xffffffffu, o2, jl);
        if (lane == 0) { wst[2 * k] = o1; wst[2 * k + 1] = o2; }
        // S3 fix-up
        const float4* __restrict__ G = reinterpret_cast<const float4*>(T + kOffG);
#pragma unroll
        for (int i = 0; i < kL; i += 2) {
            if (GEN && i >= len) break;
            const float4 g = G[i >> 1];
            x[i] = fmaf(g.x, a, fmaf(g.y, b, x[i]));
            x[i + 1] = fmaf(g.z, a, fmaf(g.w, b, x[i + 1]));
        }
    }

    if (p.filt)
        stage_out<GEN>(x, p.filt + (long long)ch * p.out_pitch + t0, buf, lane, vec4, len, n_valid,
                       p.tail_magic);

    // ---- S4..S6: energy, the two averages, ratio --------------------------------------------
    const float* __restrict__ AV = stab + p.n_sec * kSecStride;
    const float as = AV[0], al = AV[1];
    float vs = 0.0f, vl = 0.0f;
#pragma unroll
    for (int i = 0; i < kL; ++i) {
        if (GEN && i >= len) break;
        const float e = x[i] * x[i];
        x[i] = e;
        if (!GEN || i < mylen) { vs = fmaf(as, vs, e); vl = fmaf(al, vl, e); }
    }
    const float Ms = wst[2 * p.n_sec], Ml = wst[2 * p.n_sec + 1];
    const float* __restrict__ bs = GEN ? tt.beta_s : AV + 4;
    const float* __restrict__ bl = GEN ? tt.beta_l : AV + 9;
    float ws = vs, wl = vl;
    if (lane == 0) { ws += fmaf(-bs[0], Ms, Ms); wl += fmaf(-bl[0], Ml, Ml); }
    scan1(ws, bs, lane);
    scan1(wl, bl, lane);
    float ms = __shfl_up_sync(0xffffffffu, ws, 1);
    float ml = __shfl_up_sync(0xffffffffu, wl, 1);
    if (lane == 0) { ms = Ms; ml = Ml; }
    float os, ol;
    if (!GEN) { os = ws; ol = wl; }
    else { os = vs + fmaf(-tt.beta_end_s, ms, ms); ol = vl + fmaf(-tt.beta_end_l, ml, ml); }
    os = __shfl_sync(0xffffffffu, os, jl);
    ol = __shfl_sync(0xffffffffu, ol, jl);
    if (lane == 0) { wst[2 * p.n_sec] = os; wst[2 * p.n_sec + 1] = ol; }

    if (p.cf) {
        // warm-up (reading R10): samples whose global index is < lta_len give cf = 0
        const long long rem = (long long)p.lta_len - (long long)(g0 + (unsigned long long)t0);
        const int wm = rem <= 0 ? 0 : (rem > (1 << 30) ? (1 << 30) : (int)rem);
        const int base = lane * len;
        const float ratio = p.ratio, thr = p.lta_thr;
        if (wm == 0) {
#pragma unroll
            for (int i = 0; i < kL; ++i) {
                if (GEN && i >= len) break;
                const float e = x[i];
                ms = fmaf(as, ms, e); ml = fmaf(al, ml, e);
                x[i] = ml > thr ? ratio * __fdividef(ms, ml) : 0.0f;
            }
        } else {
#pragma unroll
            for (int i = 0; i < kL; ++i) {
                if (GEN && i >= len) break;
                const float e = x[i];
                ms = fmaf(as, ms, e); ml = fmaf(al, ml, e);
                x[i] = (ml > thr && base + i >= wm) ? ratio * __fdividef(ms, ml) : 0.0f;
            }
        }
        stage_out<GEN>(x, p.cf + (long long)ch * p.out_pitch + t0, buf, lane, vec4, len, n_valid,
                       p.tail_magic);
    }
    __syncwarp();
}

// The last CTA to finish advances the stream's sample counter (all CTAs read it at start).
__device__ __forceinline__ void finish_push(const PushParams& p)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(&p.ctr->ticket, 1u);
        if (t == gridDim.x - 1) {
            p.ctr->g += (unsigned long long)p.n_t;
            p.ctr->ticket = 0u;
            __threadfence();
        }
    }
}

// Channel-major push: grid = ceil(n_ch / kWarps), block = kWarps * 32.
__global__ void __launch_bounds__(kWarps * 32)
filark_push_cm_kernel(const __grid_constant__ PushParams p, const __grid_constant__ TailTab tt)
{
    extern __shared__ __align__(16) float smem[];
    const int tab_floats = p.n_sec * kSecStride + kAvgFloats;
    float* stab = smem;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int st_floats = (2 * p.n_sec + 2 + 3) & ~3;
    float* buf = smem + ((tab_floats + 3) & ~3) + warp * (32 * kPitch + st_floats);
    float* wst = buf + 32 * kPitch;
    for (int i = threadIdx.x; i < tab_floats; i += blockDim.x) stab[i] = p.tab[i];
    const unsigned long long g0 = p.ctr->g;
    __syncthreads();

    const int ch = blockIdx.x * kWarps + warp;
    if (ch < p.n_ch) {
        const int ns = 2 * p.n_sec + 2;
        float* gst = p.state + (long long)ch * ns;
        if (lane < ns) wst[lane] = gst[lane];
        if (lane + 32 < ns) wst[lane + 32] = gst[lane + 32];
        __syncwarp();
        long long t0 = 0;
        for (int tile = 0; tile < p.n_full; ++tile, t0 += kTile)
            process_tile<false>(p, tt, stab, buf, wst, ch, t0, lane, g0);
        if (p.tail_len > 0)
            process_tile<true>(p, tt, stab, buf, wst, ch, t0, lane, g0);
        __syncwarp();
        if (lane < ns) gst[lane] = wst[lane];
        if (lane + 32 < ns) gst[lane + 32] = wst[lane + 32];
    }
    finish_push(p);
}

// Diagnostic kernel (FILARK_FLAG_SERIAL_SCAN): one thread per channel, serial in time, the same
// state-space sections and the same state layout, no blocked scan.  Element (c, t) of a chunk
// is at c * sc + t * st.
__global__ void __launch_bounds__(128)
filark_push_serial_kernel(const __grid_constant__ PushParams p, long long sc_in, long long st_in,
                          long long sc_out, long long st_out, long long state_sc, long long state_sk)
{
    extern __shared__ __align__(16) float smem[];
    const int tab_floats = p.n_sec * kSecStride + kAvgFloats;
    for (int i = threadIdx.x; i < tab_floats; i += blockDim.x) smem[i] = p.tab[i];
    const unsigned long long g0 = p.ctr->g;
    __syncthreads();
    const int ch = blockIdx.x * blockDim.x + threadIdx.x;
    if (ch < p.n_ch) {
        float s[2 * kMaxSec + 2];
        const int ns = 2 * p.n_sec + 2;
        for (int i = 0; i < ns; ++i) s[i] = p.state[ch * state_sc + i * state_sk];
        const float* AV = smem + p.n_sec * kSecStride;
        const float cs = AV[2], cl = AV[3];
        float ms = s[ns - 2], ml = s[ns - 1];
        for (long long t = 0; t < p.n_t; ++t) {
            float v = p.in[ch * sc_in + t * st_in] * p.gain;
            for (int k = 0; k < p.n_sec; ++k) {
                const float* T = smem + k * kSecStride;
                const float q0 = T[1], q1 = T[2], q2 = T[3], q3 = T[4], q4 = T[5];
                const float s1 = s[2 * k], s2 = s[2 * k + 1];
                float y;
                if (__float_as_int(T[0]) == kKindR) {
                    y = fmaf(q2, s1, fmaf(q3, s2, v));
                    s[2 * k] = fmaf(q0, s1, fmaf(q1, s2, v));
                    s[2 * k + 1] = fmaf(q0, s2, -q1 * s1);
                } else {
                    y = fmaf(q0, v, s1);
                    s[2 * k] = fmaf(q3, y, fmaf(q1, v, s2));
                    s[2 * k + 1] = fmaf(q4, y, q2 * v);
                }
                v = y;
            }
            if (p.filt) p.filt[ch * sc_out + t * st_out] = v;
            const float e = v * v;
            ms = fmaf(-cs, ms, ms) + e;
            ml = fmaf(-cl, ml, ml) + e;
            if (p.cf)
                p.cf[ch * sc_out + t * st_out] =
                    (ml > p.lta_thr && g0 + (unsigned long long)t >= (unsigned long long)p.lta_len)
                        ? p.ratio * __fdividef(ms, ml) : 0.0f;
        }
        s[ns - 2] = ms; s[ns - 1] = ml;
        for (int i = 0; i < ns; ++i) p.state[ch * state_sc + i * state_sk] = s[i];
    }
    finish_push(p);
}

}  // namespace filark
