// filark_kernels.cuh -- sm_100a kernels of the fused SOS + STA/LTA stream path.
//
// Steps (include/filark_stream.h): S0 load, S1 per-section local scan,
// S2 warp-shuffle combine, S3 fix-up + carried state, S4 energy, S5 STA/LTA scans,
// S6 ratio + warm-up, S7 store.  One launch per push; the chunk is read once from HBM and
// each output is written once.
//
// Channel-major mapping (time contiguous): one warp owns one channel.  The time axis of a push
// is cut into sub-blocks of L samples ("slots"); a tile is 64 consecutive slots, and lane l
// owns slots 2l and 2l+1 of the tile as the two halves of packed f32x2 registers, so every
// arithmetic instruction of the recurrences is an FFMA2 working on two sub-blocks at once.
// A lane's samples stay in registers through every section and the STA/LTA.  Tiles of a channel
// are processed in time order by the same warp; the carried state sits in shared memory between
// tiles and in global memory between pushes.
//
// Ragged pushes need no second code path: slots are aligned to the END of the push, the first
// slot is the short one (r <= L samples, zero-padded at its front -- a zero-state recurrence
// stays at rest through leading zeros), and it always sits in the high half of lane 0 of tile 0
// (one idle slot in front of it when r < L), so that its shifted fix-up table is a per-lane
// table pointer.  Trailing idle slots hold zeros and are never stored.
//
// The recurrences are exact restatements of the oracle's definition:
//   section:  s[n] = A s[n-1] + B x[n],  y[n] = C s[n-1] + D x[n]           (design.hpp)
//   slot with carry-in s_in, local pass from zero state giving y_loc and end state v:
//             y[i] = y_loc[i] + (C A^i) s_in,   s_out = A^len s_in + v
//   averages: m~[n] = alpha m~[n-1] + e[n]  (m~ = m * N),  cf = (N_l/N_s) s~/l~
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace filark {

constexpr int kWarps = 4;              // warps (= channels in flight) per CTA
constexpr int kMaxSec = 16;
constexpr int kSteps = 5;              // log2(32) scan steps
constexpr int kKindDF2 = 0, kKindDF2G = 1, kKindDelta = 2, kKindDeltaG = 3, kKindNormal = 4;

// ---- device table of one sub-block length L (floats); see build_variant_table() ----------------
// per section, stride SecTab<L>::stride:
//   [0] kind (int bits)  [1..5] local-pass coefficients  [7] scan steps needed (int bits)
//   [8..11]  P = A^L                       [12..31] Q[d] = A^(2L 2^d), d = 0..4 (row-major 2x2)
//   [32 ..)  Apow[r] = A^r, r = 0..L       (carry across the short first slot)
//   G0: 2L rows (g1, g2): rows -L..-1 are zero, row i >= 0 is C A^i     (+ 4 floats pad)
//   G1: the same shifted down by one row (row j holds G0 row j-1): 16-byte aligned odd shifts
// after the sections, the averages block AvgTab<L> (STA then LTA interleaved where paired):
//   [0] alpha_s [1] alpha_l
//   [2..3] 1 - alpha^L  [4..13] 1 - alpha^(2L 2^d) (s,l interleaved)  [14] 1/N_s [15] 1/N_l
//   [16 ..) 1 - alpha^r, r = 0..L (s,l interleaved)   then alpha^-sh, sh = 0..L-1 (s,l interleaved)
template <int L> struct SecTab {
    static constexpr int apow = 32;
    static constexpr int g0 = apow + 4 * (L + 1);
    static constexpr int gsz = 4 * L + 4;
    static constexpr int g1 = g0 + gsz;
    static constexpr int stride = g1 + gsz;
};
template <int L> struct AvgTab {
    static constexpr int beta_l = 2, beta_q = 4, beta_r = 16;
    static constexpr int inv = beta_r + 2 * (L + 1);
    static constexpr int size = (inv + 2 * L + 3) & ~3;
};
constexpr int kOffKind = 0, kOffCoef = 1, kOffNSteps = 7, kOffP = 8, kOffQ = 12;

struct Counter { unsigned long long g; unsigned int ticket; unsigned int pad; };

struct PushParams {
    const float* in;
    float* filt;
    float* cf;
    const float* tab;        // table of the chosen L (device)
    float* state;            // channel-major: [n_ch][2 n_sec + 2]; time-major: [2 n_sec + 2][n_ch]
    Counter* ctr;
    long long n_t, in_pitch, out_pitch;
    int n_ch, n_sec;
    int n_tiles;             // tiles per channel
    int lead;                // idle slots in front of the first one (0, or 1 when r < L)
    int r;                   // samples in the first slot, 1..L
    int pad0;                // zeros in front of sample 0: lead L + (L - r)
    int last_lane, last_half;// lane / half of the slot holding the last sample (in the last tile)
    int lta_len;
    int vec4;                // float4 global accesses are legal (alignment, pitch, n_t % 4 == 0)
    float gain, ratio, lta_thr;
};

__device__ __forceinline__ float ld_stream(const float* p) { return __ldcs(p); }
__device__ __forceinline__ float4 ld_stream4(const float* p) { return __ldcs(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ void st_stream(float* p, float v) { __stcs(p, v); }
__device__ __forceinline__ void st_stream4(float* p, float4 v) { __stcs(reinterpret_cast<float4*>(p), v); }

__device__ __forceinline__ float rcp_fast(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 fma2(float a, float2 b, float2 c) { return __ffma2_rn(make_float2(a, a), b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 shfl_up2(float2 v, int d) {
    return make_float2(__shfl_up_sync(0xffffffffu, v.x, d), __shfl_up_sync(0xffffffffu, v.y, d));
}
__device__ __forceinline__ float2 shfl2(float2 v, int src) {
    return make_float2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}

template <int L> struct Geo {
    static constexpr int pitch = 2 * L + 4;        // floats per lane region: LDS.128 conflict-free
    static constexpr int tile = 64 * L;            // samples per tile
    static constexpr int buf_floats = 32 * pitch;
};

// S0: bring one tile of one channel into packed registers: x[i] = (slot 2l sample i, slot 2l+1
// sample i).  t0 = time index (within the push) of the tile's padded position 0; samples outside
// [0, n_t) read as zero.
template <int L>
__device__ __forceinline__ void stage_in(float2 (&x)[L], const float* __restrict__ src, float* buf,
                                         int lane, bool vec4, long long t0, long long n_t, float gain)
{
    constexpr int P = Geo<L>::pitch;
    if (vec4) {
        constexpr int C = L / 4;                   // float4 per slot
        float4 e[C], o[C];
        const bool inside = t0 >= 0 && t0 + Geo<L>::tile <= n_t;
#pragma unroll
        for (int m = 0; m < C; ++m) {
            const int k = 32 * m + lane, j = k / C, q = k - j * C;
            const long long te = t0 + 2 * j * L + 4 * q, to = te + L;
            e[m] = (inside || (te >= 0 && te < n_t)) ? ld_stream4(src + te) : make_float4(0.f, 0.f, 0.f, 0.f);
            o[m] = (inside || (to >= 0 && to < n_t)) ? ld_stream4(src + to) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int m = 0; m < C; ++m) {
            const int k = 32 * m + lane, j = k / C, q = k - j * C;
            float* d = buf + j * P + 8 * q;
            *reinterpret_cast<float4*>(d) = make_float4(e[m].x, o[m].x, e[m].y, o[m].y);
            *reinterpret_cast<float4*>(d + 4) = make_float4(e[m].z, o[m].z, e[m].w, o[m].w);
        }
    } else {
#pragma unroll 8
        for (int m = 0; m < 2 * L; ++m) {
            const int el = 32 * m + lane, slot = el / L, i = el - slot * L;
            const long long t = t0 + el;
            const float v = (t >= 0 && t < n_t) ? ld_stream(src + t) : 0.0f;
            buf[(slot >> 1) * P + 2 * i + (slot & 1)] = v;
        }
    }
    __syncwarp();
    const float2 g2 = f2(gain);
#pragma unroll
    for (int q = 0; q < L / 2; ++q) {
        const float4 v = *reinterpret_cast<const float4*>(buf + lane * P + 4 * q);
        x[2 * q] = mul2(make_float2(v.x, v.y), g2);
        x[2 * q + 1] = mul2(make_float2(v.z, v.w), g2);
    }
    __syncwarp();
}

// S7: packed registers -> one output array, same geometry as stage_in.
template <int L>
__device__ __forceinline__ void stage_out(const float2 (&x)[L], float* __restrict__ dst, float* buf,
                                          int lane, bool vec4, long long t0, long long n_t)
{
    constexpr int P = Geo<L>::pitch;
#pragma unroll
    for (int q = 0; q < L / 2; ++q)
        *reinterpret_cast<float4*>(buf + lane * P + 4 * q) =
            make_float4(x[2 * q].x, x[2 * q].y, x[2 * q + 1].x, x[2 * q + 1].y);
    __syncwarp();
    if (vec4) {
        constexpr int C = L / 4;
        const bool inside = t0 >= 0 && t0 + Geo<L>::tile <= n_t;
#pragma unroll
        for (int m = 0; m < C; ++m) {
            const int k = 32 * m + lane, j = k / C, q = k - j * C;
            const float* s = buf + j * P + 8 * q;
            const float4 a = *reinterpret_cast<const float4*>(s);
            const float4 b = *reinterpret_cast<const float4*>(s + 4);
            const long long te = t0 + 2 * j * L + 4 * q, to = te + L;
            if (inside || (te >= 0 && te < n_t)) st_stream4(dst + te, make_float4(a.x, a.z, b.x, b.z));
            if (inside || (to >= 0 && to < n_t)) st_stream4(dst + to, make_float4(a.y, a.w, b.y, b.w));
        }
    } else {
#pragma unroll 8
        for (int m = 0; m < 2 * L; ++m) {
            const int el = 32 * m + lane, slot = el / L, i = el - slot * L;
            const long long t = t0 + el;
            const float v = buf[(slot >> 1) * P + 2 * i + (slot & 1)];
            if (t >= 0 && t < n_t) st_stream(dst + t, v);
        }
    }
    __syncwarp();
}

// One tile of one channel: S0..S7.
template <int L>
__device__ __forceinline__ void process_tile(const PushParams& p, const float* __restrict__ stab,
                                             float* buf, float* wst, int ch, int tile, int lane,
                                             unsigned long long g0)
{
    using ST = SecTab<L>;
    using AT = AvgTab<L>;
    const bool vec4 = p.vec4 != 0;
    const bool first = tile == 0, last = tile == p.n_tiles - 1;
    const long long t0 = (long long)tile * Geo<L>::tile - p.pad0;
    // the slot that receives the carried state: low half of lane 0, except in tile 0 of a ragged
    // push, where it is the (short) high half behind one idle slot
    const bool inj_hi = first && p.lead != 0;
    const int r = first ? p.r : L;                 // samples in that slot
    const int sh = L - r;                          // its fix-up rows are shifted down by sh
    const int jl = last ? p.last_lane : 31;
    const bool out_hi = last ? p.last_half != 0 : true;
    // per-lane fix-up table offset (floats) inside a section's table
    int goff = ST::g0 + 2 * L;
    if (lane == 0 && sh != 0) goff = (sh & 1) ? ST::g1 + 2 * (L - sh + 1) : ST::g0 + 2 * (L - sh);
    const float m_lo = (lane == 0 && !inj_hi) ? 1.0f : 0.0f;
    const float m_hi = (lane == 0 && inj_hi) ? 1.0f : 0.0f;

    float2 x[L];
    stage_in<L>(x, p.in + (long long)ch * p.in_pitch, buf, lane, vec4, t0, p.n_t, p.gain);

    // ---- S1..S3 per section -------------------------------------------------------------------
    for (int k = 0; k < p.n_sec; ++k) {
        const float* __restrict__ T = stab + k * ST::stride;
        const int kind = __float_as_int(T[kOffKind]);
        const float c0 = T[kOffCoef], c1 = T[kOffCoef + 1], c2 = T[kOffCoef + 2], c3 = T[kOffCoef + 3];
        float2 v1 = f2(0.0f), v2 = f2(0.0f);       // packed state: .x = low slot, .y = high slot
        if (kind == kKindDF2) {
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 w = fma2(c0, v1, fma2(c1, v2, x[i]));
                x[i] = fma2(c2, v1, fma2(c3, v2, w));
                v2 = v1; v1 = w;
            }
        } else if (kind == kKindDelta) {
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 u = fma2(c0, v1, fma2(c1, v2, x[i]));
                x[i] = fma2(c2, v1, u);
                v2 = add2(v2, u); v1 = u;
            }
        } else if (kind == kKindDeltaG) {
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 u = fma2(c0, v1, fma2(c1, v2, x[i]));
                x[i] = fma2(c3, v2, fma2(c2, v1, u));
                v2 = add2(v2, u); v1 = u;
            }
        } else if (kind == kKindNormal) {
            const float2 nc1 = f2(-c1);
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 xi = x[i];
                x[i] = fma2(c2, v1, fma2(c3, v2, xi));
                const float2 n1 = fma2(c0, v1, fma2(c1, v2, xi));
                v2 = fma2(c0, v2, mul2(nc1, v1));
                v1 = n1;
            }
        } else {                                   // kKindDF2G: explicit b0 = T[kOffCoef + 4]
            const float c4 = T[kOffCoef + 4];
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 w = fma2(c0, v1, fma2(c1, v2, x[i]));
                x[i] = fma2(c2, v1, fma2(c3, v2, mul2(f2(c4), w)));
                v2 = v1; v1 = w;
            }
        }

        // S2: end states of the two slots, carried state S into its slot, scan over lane pairs
        const float S1 = wst[2 * k], S2 = wst[2 * k + 1];
        const float4 Pm = *reinterpret_cast<const float4*>(T + kOffP);          // A^L
        const float4 Ar = *reinterpret_cast<const float4*>(T + ST::apow + 4 * r);  // A^r
        const float i1 = fmaf(Ar.x, S1, Ar.y * S2), i2 = fmaf(Ar.z, S1, Ar.w * S2);
        float lo1 = fmaf(m_lo, i1, v1.x), lo2 = fmaf(m_lo, i2, v2.x);          // state after low slot (from rest)
        float hi1 = fmaf(m_hi, i1, v1.y), hi2 = fmaf(m_hi, i2, v2.y);
        // pair total W = P lo + hi, packed as (W1, W2)
        float2 W = make_float2(fmaf(Pm.x, lo1, fmaf(Pm.y, lo2, hi1)), fmaf(Pm.z, lo1, fmaf(Pm.w, lo2, hi2)));
        const int nsteps = __float_as_int(T[kOffNSteps]);
#pragma unroll
        for (int d = 0; d < kSteps; ++d) {
            if (d < nsteps) {
                const float4 Q = *reinterpret_cast<const float4*>(T + kOffQ + 4 * d);
                const float2 U = shfl_up2(W, 1 << d);
                if (lane >= (1 << d))
                    W = fma2(make_float2(Q.x, Q.z), f2(U.x), fma2(make_float2(Q.y, Q.w), f2(U.y), W));
            }
        }
        float2 E = shfl_up2(W, 1);                 // state entering the lane's low slot
        if (lane == 0) E = f2(0.0f);
        // carry-in of the high slot: P E + lo
        float o1 = fmaf(Pm.x, E.x, fmaf(Pm.y, E.y, lo1)), o2 = fmaf(Pm.z, E.x, fmaf(Pm.w, E.y, lo2));
        // new carried state: state after the slot holding the push's last sample
        float n1 = out_hi ? W.x : o1, n2 = out_hi ? W.y : o2;
        n1 = __shfl_sync(0xffffffffu, n1, jl); n2 = __shfl_sync(0xffffffffu, n2, jl);
        if (lane == 0) {
            wst[2 * k] = n1; wst[2 * k + 1] = n2;
            if (inj_hi) { o1 = S1; o2 = S2; } else { E.x = S1; E.y = S2; }
        }
        // S3 fix-up: y[i] += g1[i] ca + g2[i] cb, packed over the two slots
        const float2 ca = make_float2(E.x, o1), cb = make_float2(E.y, o2);
        const float4* __restrict__ G = reinterpret_cast<const float4*>(T + goff);
#pragma unroll
        for (int i = 0; i < L; i += 2) {
            const float4 g = G[i >> 1];
            x[i] = fma2(g.x, ca, fma2(g.y, cb, x[i]));
            x[i + 1] = fma2(g.z, ca, fma2(g.w, cb, x[i + 1]));
        }
    }

    if (p.filt)
        stage_out<L>(x, p.filt + (long long)ch * p.out_pitch, buf, lane, vec4, t0, p.n_t);

    // ---- S4..S6: energy, the two averages, ratio --------------------------------------------
    const float* __restrict__ AV = stab + p.n_sec * ST::stride;
    const float as = AV[0], al = AV[1];
    float2 vs = f2(0.0f), vl = f2(0.0f);
#pragma unroll
    for (int i = 0; i < L; ++i) {
        const float2 e = mul2(x[i], x[i]);
        x[i] = e;
        vs = fma2(as, vs, e); vl = fma2(al, vl, e);
    }
    const float Ms = wst[2 * p.n_sec], Ml = wst[2 * p.n_sec + 1];
    // carried averages into their slot: + alpha^r M = M - beta_r M
    const float bs_r = AV[AT::beta_r + 2 * r], bl_r = AV[AT::beta_r + 2 * r + 1];
    const float is = fmaf(-bs_r, Ms, Ms), il = fmaf(-bl_r, Ml, Ml);
    // packed (sta, lta) from here on
    float2 lo = make_float2(fmaf(m_lo, is, vs.x), fmaf(m_lo, il, vl.x));
    float2 hi = make_float2(fmaf(m_hi, is, vs.y), fmaf(m_hi, il, vl.y));
    const float2 bL = *reinterpret_cast<const float2*>(AV + AT::beta_l);
    float2 W = add2(hi, fma2(make_float2(-bL.x, -bL.y), lo, lo));              // alpha^L lo + hi
#pragma unroll
    for (int d = 0; d < kSteps; ++d) {
        const float2 bq = *reinterpret_cast<const float2*>(AV + AT::beta_q + 2 * d);
        const float2 U = shfl_up2(W, 1 << d);
        if (lane >= (1 << d)) W = add2(W, fma2(make_float2(-bq.x, -bq.y), U, U));
    }
    float2 E = shfl_up2(W, 1);
    if (lane == 0) E = f2(0.0f);
    float2 O = add2(lo, fma2(make_float2(-bL.x, -bL.y), E, E));                // carry-in of the high slot
    float2 N = out_hi ? W : O;
    N = shfl2(N, jl);
    if (lane == 0) {
        wst[2 * p.n_sec] = N.x; wst[2 * p.n_sec + 1] = N.y;
        // the short slot starts its second pass sh zeros early: M alpha^-sh decays to M on them
        const float2 Mv = make_float2(Ms * AV[AT::inv + 2 * sh], Ml * AV[AT::inv + 2 * sh + 1]);
        if (inj_hi) O = Mv; else E = Mv;
    }

    if (p.cf) {
        float2 ms = make_float2(E.x, O.x), ml = make_float2(E.y, O.y);
        // warm-up (reading R10): samples whose global index is < lta_len give cf = 0
        const long long rem = (long long)p.lta_len - (long long)g0 - t0;     // first padded position with cf != 0
        const float ratio = p.ratio, thr = p.lta_thr;
        if (rem <= 0) {
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 e = x[i];
                ms = fma2(as, ms, e); ml = fma2(al, ml, e);
                const float2 q = mul2(mul2(ms, f2(ratio)), make_float2(rcp_fast(ml.x), rcp_fast(ml.y)));
                x[i] = make_float2(ml.x > thr ? q.x : 0.0f, ml.y > thr ? q.y : 0.0f);
            }
        } else {
            const int wm = rem > (1 << 30) ? (1 << 30) : (int)rem;
            const int base = 2 * lane * L;
#pragma unroll
            for (int i = 0; i < L; ++i) {
                const float2 e = x[i];
                ms = fma2(as, ms, e); ml = fma2(al, ml, e);
                const float2 q = mul2(mul2(ms, f2(ratio)), make_float2(rcp_fast(ml.x), rcp_fast(ml.y)));
                x[i] = make_float2((ml.x > thr && base + i >= wm) ? q.x : 0.0f,
                                   (ml.y > thr && base + L + i >= wm) ? q.y : 0.0f);
            }
        }
        stage_out<L>(x, p.cf + (long long)ch * p.out_pitch, buf, lane, vec4, t0, p.n_t);
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

template <int L> constexpr int cm_regs_hint() { return L >= 48 ? 2 : (L >= 32 ? 3 : 4); }      // CTAs per SM to aim for

// Channel-major push: grid = ceil(n_ch / kWarps), block = kWarps * 32.
template <int L>
__global__ void __launch_bounds__(kWarps * 32, cm_regs_hint<L>())
filark_push_cm_kernel(const __grid_constant__ PushParams p)
{
    extern __shared__ __align__(16) float smem[];
    const int tab_floats = p.n_sec * SecTab<L>::stride + AvgTab<L>::size;
    float* stab = smem;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int st_floats = (2 * p.n_sec + 2 + 3) & ~3;
    float* buf = smem + tab_floats + warp * (Geo<L>::buf_floats + st_floats);
    float* wst = buf + Geo<L>::buf_floats;
    for (int i = threadIdx.x; i < tab_floats / 4; i += blockDim.x)
        reinterpret_cast<float4*>(stab)[i] = reinterpret_cast<const float4*>(p.tab)[i];
    const unsigned long long g0 = p.ctr->g;
    __syncthreads();

    const int ch = blockIdx.x * kWarps + warp;
    if (ch < p.n_ch) {
        const int ns = 2 * p.n_sec + 2;
        float* gst = p.state + (long long)ch * ns;
        if (lane < ns) wst[lane] = gst[lane];
        if (lane + 32 < ns) wst[lane + 32] = gst[lane + 32];
        __syncwarp();
        for (int tile = 0; tile < p.n_tiles; ++tile)
            process_tile<L>(p, stab, buf, wst, ch, tile, lane, g0);
        __syncwarp();
        if (lane < ns) gst[lane] = wst[lane];
        if (lane + 32 < ns) gst[lane + 32] = wst[lane + 32];
    }
    finish_push(p);
}

// Diagnostic kernel (FILARK_FLAG_SERIAL_SCAN; also the time-major path for now): one thread per
// channel, serial in time, the same state-space sections and the same state layout, no blocked
// scan.  Element (c, t) of a chunk is at c * sc + t * st.  tab = table of any L (only the
// coefficients and alphas are read); sec_stride / avg offset passed by the host.
__global__ void __launch_bounds__(128)
filark_push_serial_kernel(const __grid_constant__ PushParams p, int sec_stride, long long sc_in,
                          long long st_in, long long sc_out, long long st_out, long long state_sc,
                          long long state_sk)
{
    __shared__ float coef[kMaxSec][8];
    __shared__ float cinv[2];
    for (int i = threadIdx.x; i < p.n_sec * 8; i += blockDim.x)
        coef[i >> 3][i & 7] = p.tab[(i >> 3) * sec_stride + (i & 7)];
    if (threadIdx.x < 2) cinv[threadIdx.x] = p.tab[p.n_sec * sec_stride + 14 + threadIdx.x];
    const unsigned long long g0 = p.ctr->g;
    __syncthreads();
    const int ch = blockIdx.x * blockDim.x + threadIdx.x;
    if (ch < p.n_ch) {
        float s[2 * kMaxSec + 2];
        const int ns = 2 * p.n_sec + 2;
        for (int i = 0; i < ns; ++i) s[i] = p.state[ch * state_sc + i * state_sk];
        const float cs = cinv[0], cl = cinv[1];
        float ms = s[ns - 2], ml = s[ns - 1];
        for (long long t = 0; t < p.n_t; ++t) {
            float v = p.in[ch * sc_in + t * st_in] * p.gain;
            for (int k = 0; k < p.n_sec; ++k) {
                const float* T = coef[k];
                const int kind = __float_as_int(T[kOffKind]);
                const float c0 = T[1], c1 = T[2], c2 = T[3], c3 = T[4], c4 = T[5];
                const float s1 = s[2 * k], s2 = s[2 * k + 1];
                float y;
                if (kind == kKindDF2 || kind == kKindDF2G) {
                    const float w = fmaf(c0, s1, fmaf(c1, s2, v));
                    y = fmaf(c2, s1, fmaf(c3, s2, kind == kKindDF2 ? w : c4 * w));
                    s[2 * k + 1] = s1; s[2 * k] = w;
                } else if (kind == kKindDelta || kind == kKindDeltaG) {
                    const float u = fmaf(c0, s1, fmaf(c1, s2, v));
                    y = fmaf(c2, s1, u);
                    if (kind == kKindDeltaG) y = fmaf(c3, s2, y);
                    s[2 * k + 1] = s2 + u; s[2 * k] = u;
                } else {
                    y = fmaf(c2, s1, fmaf(c3, s2, v));
                    s[2 * k] = fmaf(c0, s1, fmaf(c1, s2, v));
                    s[2 * k + 1] = fmaf(c0, s2, -c1 * s1);
                }
                v = y;
            }
            if (p.filt) p.filt[ch * sc_out + t * st_out] = v;
            const float e = v * v;
            ms = fmaf(-cs, ms, ms) + e;      // (1 - 1/N) m~ + e without rounding 1 - 1/N (reading R13)
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
